"""The allocation-free entry point (include/lcf_noalloc.h): lcf_gram_global_noalloc against the plan path's covariance of
the same data (one all-ones window, precision 1: lcf_get_gram), two calls in a row on the shared scratch array.  Collected
last on purpose (the suite runs with pytest -x)."""
import ctypes as C
import re
from pathlib import Path

import numpy as np
import pytest

from paper_2405_11105_b200 import synth

ROOT = Path(__file__).resolve().parents[1]
GRAM_TOL = 1e-12           # the Gram gate of tests/test_gpu_parity.py at precision 1 (relative to max |R|)


def test_noalloc_symbols_are_exported():
    from paper_2405_11105_b200 import build, lcf, lcf_noalloc
    build.build()
    header = re.sub(r"/\*.*?\*/", "", (ROOT / "include" / "lcf_noalloc.h").read_text(), flags=re.S)
    declared = set(re.findall(r"\b(lcf_[a-z_]+)\s*\(", header))
    assert declared == set(lcf_noalloc.EXPORTS)
    lib = C.CDLL(str(lcf.LIB_PATH))
    for name in declared:
        assert hasattr(lib, name), f"{name} declared in include/lcf_noalloc.h but not exported"
    # argument checks come before any CUDA call: they work without a GPU and say what is wrong
    L = lcf_noalloc._lib()
    assert L.lcf_gram_global_noalloc(None, 4, 16, None, None) == lcf.ERR_INVALID_ARG
    assert L.lcf_gram_global_noalloc(C.c_void_p(256), 0, 16, C.c_void_p(256), None) == lcf.ERR_INVALID_ARG
    assert L.lcf_gram_global_noalloc(C.c_void_p(256), lcf_noalloc.MAX_FRAMES + 1, 16, C.c_void_p(256), None) == lcf.ERR_UNSUPPORTED
    assert "at most 128 frames" in lcf_noalloc.last_error()
    assert L.lcf_gram_global_noalloc(C.c_void_p(256), 4, (1 << 30) + 1, C.c_void_p(256), None) == lcf.ERR_UNSUPPORTED


@pytest.mark.gpu
def test_noalloc_gram_matches_the_plan_path_twice_in_a_row():
    import torch
    assert torch.cuda.is_available(), "this test needs a CUDA device"
    from paper_2405_11105_b200 import build, lcf, lcf_noalloc
    build.build()
    lcf.load()
    # first call: the largest supported ensemble, ragged pixel count; second call: a smaller one, so that the scratch
    # array still holds the first call's partial sums around and beyond the entries the second one uses
    cases = [(96, 85, 128, 11), (37, 50, 33, 12)]
    refs, outs = [], []
    for (Nz, Nx, N, seed) in cases:
        iq = synth.random_cube(Nz, Nx, N, seed=seed)
        iq_d = torch.from_numpy(iq).cuda()
        f = synth.FilterSpec(1, 1, 0.0, 0.0, 0.0, synth.HARD_FIXED, k_fixed=1, precision=1)     # one all-ones window, fp64 Gram
        pd_d = torch.empty((Nx, Nz), dtype=torch.float32, device="cuda")
        with lcf.Plan.from_spec(Nz, Nx, N, f) as plan:
            plan.filter(iq_d, pd_d)
            torch.cuda.synchronize()
            refs.append(plan.gram()[0])
        outs.append((iq_d, N, Nx * Nz, torch.full((N, N), float("nan"), dtype=torch.complex128, device="cuda")))
    torch.cuda.synchronize()
    st = torch.cuda.current_stream()
    for iq_d, N, P, R_d in outs:                              # back to back on one stream, no synchronisation in between
        lcf_noalloc.gram_global_noalloc(iq_d, N, P, R_d, st)
    torch.cuda.synchronize()
    for (iq_d, N, P, R_d), ref in zip(outs, refs):
        R = R_d.cpu().numpy()
        assert np.isfinite(R.view(np.float64)).all()
        err = np.abs(R - ref).max() / np.abs(ref).max()
        assert err <= GRAM_TOL, f"N = {N}: Gram err {err:.3e}"
        assert np.abs(R - R.conj().T).max() <= GRAM_TOL * np.abs(ref).max()      # Hermitian
    # the same input again gives the same bits (fixed summation order), whatever the scratch held
    iq_d, N, P, R_d = outs[0]
    R2 = torch.empty_like(R_d)
    torch.cuda.synchronize()
    free_before = torch.cuda.mem_get_info()[0]                # (the module, with its 4 MiB array, was loaded by the first call)
    lcf_noalloc.gram_global_noalloc(iq_d, N, P, R2, st)
    torch.cuda.synchronize()
    assert torch.cuda.mem_get_info()[0] >= free_before        # the call took no device memory
    assert torch.equal(R2, R_d)
    # beyond the maximum: refused with a sentence, nothing launched
    with pytest.raises(lcf.LcfError) as ei:
        lcf_noalloc.gram_global_noalloc(iq_d, 129, 64, R_d, st)
    assert ei.value.status == lcf.ERR_UNSUPPORTED and "at most 128 frames" in str(ei.value)
