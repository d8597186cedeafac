"""CPU-only checks of the product's host side: liblcf.so builds, loads and exports every symbol
include/lcf.h declares; argument validation returns status codes (no CUDA call is made before the
arguments are validated); the library refuses to run without a GPU; the ensemble sharding used for
multi-GPU runs is a partition (world_size 2, gloo)."""
import ctypes as C
import os
import re
import subprocess
import sys
from pathlib import Path

import numpy as np
import pytest

ROOT = Path(__file__).resolve().parent.parent


@pytest.fixture(scope="module")
def lcf():
    from paper_2405_11105_b200 import build, lcf as binding
    build.build()
    binding.load()
    return binding


def test_library_exports_every_declared_symbol(lcf):
    header = (ROOT / "include" / "lcf.h").read_text()
    header = re.sub(r"/\*.*?\*/", "", header, flags=re.S)
    declared = set(re.findall(r"\b(lcf_[a-z_]+)\s*\(", header))
    assert {"lcf_plan_create", "lcf_filter", "lcf_plan_destroy"} <= declared
    lib = C.CDLL(str(lcf.LIB_PATH))
    for name in sorted(declared):
        assert hasattr(lib, name), f"{name} declared in include/lcf.h but not exported"
    assert declared == set(lcf.EXPORTS)


def test_status_strings(lcf):
    seen = {lcf.status_string(s) for s in range(6)}
    assert len(seen) == 6 and "ok" in seen
    assert lcf.status_string(99) == "unknown status"


def _create(lcf, Nz=8, Nx=8, N=4, Kz=1, Kx=1, sz=0.0, sx=0.0, tr=0.0, mode=0, k=1, frac=0.995, beta=0.5, prec=0, cs=1.0):
    L = lcf.load()
    h = C.c_void_p(None)
    w = lcf.Windows(Kz, Kx, sz, sx, tr)
    t = lcf.Thresh(mode, k, frac, beta, prec, cs)
    st = L.lcf_plan_create(C.byref(h), Nz, Nx, N, C.byref(w), C.byref(t))
    return st, h


@pytest.mark.parametrize("kw", [
    dict(Nz=0), dict(Nx=-1), dict(N=1), dict(Kz=0), dict(Kx=0), dict(mode=17), dict(mode=-1), dict(mode=15, k=-1), dict(mode=16, frac=1.5), dict(mode=14, beta=0.0), dict(mode=11, cs=0.0), dict(mode=12, beta=0.0), dict(mode=8, beta=0.0), dict(mode=9, cs=0.0), dict(mode=10, cs=-2.0), dict(mode=10, beta=0.0), dict(mode=4, cs=0.0), dict(mode=5, cs=-1.0), dict(mode=6, cs=0.0),
    dict(k=-1), dict(k=5), dict(mode=1, frac=1.0), dict(mode=3, frac=0.0), dict(mode=2, beta=0.0),
    dict(prec=2), dict(sz=float("nan")), dict(tr=float("inf")),
])
def test_invalid_arguments_are_refused(lcf, kw):
    st, h = _create(lcf, **kw)
    assert st == lcf.ERR_INVALID_ARG and not h.value


def test_null_pointers(lcf):
    L = lcf.load()
    assert L.lcf_plan_create(None, 8, 8, 4, None, None) == lcf.ERR_INVALID_ARG
    assert L.lcf_plan_destroy(None) == lcf.OK
    assert L.lcf_filter(None, None, None, None) == lcf.ERR_INVALID_ARG
    assert L.lcf_num_windows(None) == 0
    assert L.lcf_measure_peak(7, None) == lcf.ERR_INVALID_ARG
    assert L.lcf_get_converged(None, None) == lcf.ERR_INVALID_ARG
    assert L.lcf_set_max_sweeps(None, 3) == lcf.ERR_INVALID_ARG


def test_header_is_plain_c_and_matches_the_binding(tmp_path):
    """include/lcf.h compiles as C without the CUDA headers (cudaStream_t is forward-declared), and the
    struct layouts the ctypes binding assumes are the compiler's."""
    from paper_2405_11105_b200 import lcf as binding
    src = tmp_path / "t.c"
    src.write_text(r"""
#include <stddef.h>
#include <stdio.h>
#include "lcf.h"
int main(void) {
    lcf_status (*f)(lcf_plan*, const void*, float*, cudaStream_t) = lcf_filter; (void)f;
    printf("%zu %zu %zu %zu %zu %zu %zu\n", sizeof(lcf_thresh), offsetof(lcf_thresh, k_fixed), offsetof(lcf_thresh, energy_frac),
           offsetof(lcf_thresh, beta), offsetof(lcf_thresh, precision), offsetof(lcf_thresh, cut_scale), sizeof(lcf_windows));
    return 0;
}
""")
    exe = tmp_path / "t"
    subprocess.run(["gcc", "-std=c99", "-Wall", "-Werror", "-I", str(ROOT / "include"), str(src), "-o", str(exe),
                    str(binding.LIB_PATH), "-Wl,-rpath," + str(binding.LIB_PATH.parent)], check=True)
    out = subprocess.run([str(exe)], capture_output=True, text=True, check=True).stdout.split()
    T = binding.Thresh
    assert [int(v) for v in out] == [C.sizeof(T), T.k_fixed.offset, T.energy_frac.offset, T.beta.offset, T.precision.offset,
                                     T.cut_scale.offset, C.sizeof(binding.Windows)]


def test_scale_exponent_of_the_tensor_path(lcf):
    """Host logic behind the fp16 split-precision kernels: amax * 2^k must land in [256, 512)."""
    import math
    for a in (1.0, 3.53, 255.9, 256.0, 511.9, 512.0, 1.37e-9, 7.7e5, 3.3e12, 6.1e-5, 65504.0, 1e-25, 1e30):
        k = lcf.scale_exponent(a)
        assert 256.0 <= math.ldexp(a, k) < 512.0, (a, k)
        assert lcf.scale_exponent(-a) == k                     # the sign bit is ignored
    for a in (0.0, float("inf"), float("nan"), 1e-40):          # nothing to scale by: zero, non-finite, denormal
        assert lcf.scale_exponent(a) == 0
    assert lcf.scale_exponent(2e-38) == 100 and lcf.scale_exponent(3e38) == -100   # clamped


def test_no_cpu_fallback(lcf):
    import torch
    if torch.cuda.is_available():
        pytest.skip("a GPU is present")
    st, h = _create(lcf)
    assert st == lcf.ERR_CUDA and not h.value            # fails loudly, does not compute on the host
    with pytest.raises(lcf.LcfError):
        lcf.Plan(8, 8, 4, 1, 1, 0.0, 0.0, 0.0, 0, 1)


def test_product_never_imports_the_oracle():
    pkg = ROOT / "paper_2405_11105_b200"
    for f in list(pkg.rglob("*.py")) + list(pkg.rglob("*.cu")) + list(pkg.rglob("*.h")):
        txt = f.read_text()
        assert "lcf_oracle" not in txt and "from oracle" not in txt and "import oracle" not in txt, f


def test_ensemble_shard_is_a_partition():
    from paper_2405_11105_b200.shard import ensemble_shard
    for n in (0, 1, 7, 16):
        for w in (1, 2, 3, 8):
            parts = [ensemble_shard(n, r, w) for r in range(w)]
            assert sorted(sum(parts, [])) == list(range(n))
            assert max(len(p) for p in parts) - min(len(p) for p in parts) <= 1
    with pytest.raises(ValueError):
        ensemble_shard(4, 2, 2)


_WORKER = r"""
import os, sys
import numpy as np, torch, torch.distributed as dist
sys.path.insert(0, os.environ["LCF_ROOT"])
from paper_2405_11105_b200.shard import ensemble_shard, gather_images
dist.init_process_group("gloo")
r, w = dist.get_rank(), dist.get_world_size()
n = 5
mine = ensemble_shard(n, r, w)
if torch.cuda.is_available():
    # real lcf_filter output: every rank filters its own ensembles (all on the one visible GPU) and
    # rank 0 checks the gathered images against filtering all of them itself
    from paper_2405_11105_b200 import lcf, synth
    def run(es):
        out = {}
        with lcf.Plan(16, 12, 8, 2, 2, 5.0, 5.0, 3.0, synth.SOFT_ENERGY) as plan:
            for e in es:
                iq = torch.from_numpy(synth.random_cube(16, 12, 8, seed=40 + e)).cuda()
                pd = torch.empty((12, 16), dtype=torch.float32, device="cuda")
                plan.filter(iq, pd)
                torch.cuda.synchronize()
                out[e] = pd.cpu()
        return out
    local = run(mine)
    imgs = gather_images(local, n)
    if r == 0:
        ref = run(range(n))
        assert all(torch.equal(imgs[e], ref[e]) for e in range(n))
else:
    local = {e: torch.full((2, 3), float(e)) for e in mine}      # no GPU here: stand-in images, the sharding logic only
    imgs = gather_images(local, n)
    assert len(imgs) == n and all(float(imgs[e][0, 0]) == e for e in range(n))
dist.barrier()
dist.destroy_process_group()
sys.stdout.write(f"rank {r} ok {mine}\n"); sys.stdout.flush()
"""


def test_two_rank_ensemble_sharding_gloo(tmp_path):
    run_two_rank_workers(tmp_path, 29571)


def run_two_rank_workers(tmp_path, port):
    script = tmp_path / "worker.py"
    script.write_text(_WORKER)
    env = dict(os.environ, LCF_ROOT=str(ROOT), MASTER_ADDR="127.0.0.1")
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node=2",
           "--master-addr", "127.0.0.1", "--master-port", str(port), str(script)]
    out = subprocess.run(cmd, env=env, capture_output=True, text=True, timeout=240)
    assert out.returncode == 0, out.stdout + out.stderr
    lines = {ln.strip() for ln in out.stdout.splitlines()}
    assert "rank 0 ok [0, 2, 4]" in lines and "rank 1 ok [1, 3]" in lines, out.stdout
