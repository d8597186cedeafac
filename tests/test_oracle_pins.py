"""Pins of the float64 oracle (oracle/lcf_oracle.c) to things other than itself.

The paper prints no reproducible worked example (its figure values need its private data), so the
oracle is pinned to what the mathematics fixes: LAPACK (numpy eigh/svd/matmul, float64), closed
forms, identities that follow from Eqs. 1-5, 9, 11-13, and a
literal brute-force implementation of the paper's own data flow (form C_w = W C explicitly, as the
paper does) on tiny inputs.  A dropped term, wrong sign, transposed or
un-conjugated operand in any oracle step fails at least one test here.
"""
import numpy as np
import pytest

from paper_2405_11105_b200 import synth


def cn(rng, shape):
    return (rng.standard_normal(shape) + 1j * rng.standard_normal(shape)) / np.sqrt(2)


def casorati(iq):
    """[N][Nx][Nz] -> C [P][N], row p = z + Nz*x."""
    N = iq.shape[0]
    return iq.reshape(N, -1).T.astype(np.complex128)


def rand_herm(rng, n, cond=1e6):
    q, _ = np.linalg.qr(cn(rng, (n, n)))
    lam = np.logspace(0, -np.log10(cond), n)
    return (q * lam) @ q.conj().T, lam, q


# ---------------------------------------------------------------- windows (Eq. 11)
def test_windows_support_lengths_config2(oracle):
    # centres 15.5 + 32 k, |d| <= 72 on a 256 axis: supports counted by hand
    g = oracle.axis_windows(256, 8, 24.0, 3.0)
    assert [(row != 0).sum() for row in g] == [88, 120, 144, 144, 144, 144, 120, 88]
    # peak of an interior window: nearest pixels are 0.5 px from the centre
    assert np.isclose(g[3].max(), np.exp(-0.25 / (2 * 24.0 ** 2)), rtol=1e-15)


def test_windows_symmetry_and_special_cases(oracle):
    for n, K, s, t in [(64, 3, 16.0, 3.0), (100, 4, 10.0, 0.0), (37, 5, 3.0, 2.0)]:
        g = oracle.axis_windows(n, K, s, t)
        assert np.allclose(g, g[::-1, ::-1], rtol=1e-12, atol=0)          # grid is mirror symmetric
        assert np.array_equal(g != 0, (g != 0)[::-1, ::-1])
        assert g.max() <= 1.0 and g.min() >= 0.0
        if t <= 0:
            assert (g > 0).all()
    assert np.array_equal(oracle.axis_windows(17, 1, 0.0, 0.0), np.ones((1, 17)))     # all-ones
    # one pixel, centred exactly: c = 0.5*1/1 - 0.5 = 0 -> weight exp(0) = 1
    assert oracle.axis_windows(1, 1, 5.0, 3.0)[0, 0] == 1.0
    # centre of a 2-window grid on 8 px: c = 1.5, 5.5; value at i=0 of window 0 = exp(-1.5^2/(2*4))
    g = oracle.axis_windows(8, 2, 2.0, 0.0)
    assert np.isclose(g[0, 0], np.exp(-2.25 / 8.0), rtol=1e-15)
    assert np.isclose(g[1, 7], np.exp(-2.25 / 8.0), rtol=1e-15)
    # truncation is inclusive: |d| = 1.5 <= trunc*sigma = 1.5 kept, 2.5 dropped
    g = oracle.axis_windows(8, 2, 1.5, 1.0)
    assert g[0, 0] > 0 and g[0, 3] > 0 and g[0, 4] == 0


# ---------------------------------------------------------------- Gram (Eqs. 1, 12)
def test_gram_matches_blas_and_identities(oracle):
    rng = np.random.default_rng(1)
    N, Nx, Nz = 7, 9, 11
    iq = cn(rng, (N, Nx, Nz)).astype(np.complex64)
    gz = oracle.axis_windows(Nz, 2, 3.0, 2.0)
    gx = oracle.axis_windows(Nx, 3, 2.0, 0.0)
    Cm = casorati(iq)
    Rsum = 0
    for kz in range(2):
        for kx in range(3):
            w = (gx[kx][:, None] * gz[kz][None, :]).reshape(-1)
            R = oracle.gram(iq, gz[kz], gx[kx])
            ref = (Cm.conj().T * w ** 2) @ Cm                       # C^H diag(w^2) C
            assert np.abs(R - ref).max() <= 1e-13 * np.abs(ref).max()
            assert np.abs(R - R.conj().T).max() == 0.0               # exactly Hermitian
            # trace(R) = sum_p w_p^2 ||s_p||^2
            assert np.isclose(np.trace(R).real, (w ** 2 * (np.abs(Cm) ** 2).sum(1)).sum(), rtol=1e-13)
            assert np.linalg.eigvalsh(R).min() >= -1e-12 * np.trace(R).real
            Rsum = Rsum + R
    wtot = sum(np.outer(gx[kx], gz[kz]).reshape(-1) ** 2 for kz in range(2) for kx in range(3))
    assert np.abs(Rsum - (Cm.conj().T * wtot) @ Cm).max() <= 1e-12 * np.abs(Rsum).max()


def test_gram_conjugation_convention(oracle):
    # R[i][j] = sum conj(S_i) S_j : for one pixel with s = (1, i) -> R[0][1] = conj(1)*i = +i
    iq = np.zeros((2, 1, 1), dtype=np.complex64)
    iq[0, 0, 0] = 1.0
    iq[1, 0, 0] = 1j
    R = oracle.gram(iq, np.ones(1), np.ones(1))
    assert R[0, 1] == 1j and R[1, 0] == -1j and R[0, 0] == 1 and R[1, 1] == 1


# ---------------------------------------------------------------- EVD (Eqs. 2, 3)
@pytest.mark.parametrize("n,cond", [(1, 1.0), (2, 10.0), (5, 1e3), (32, 1e7), (64, 1e10)])
def test_jacobi_vs_lapack(oracle, n, cond):
    rng = np.random.default_rng(n)
    A, lam_true, _ = rand_herm(rng, n, cond)
    A = (A + A.conj().T) / 2
    lam, V, sweeps = oracle.jacobi(A)
    w = np.linalg.eigvalsh(A)[::-1]
    assert np.abs(lam - w).max() <= 1e-13 * abs(w).max()
    assert (np.diff(lam) <= 0).all()                                   # sorted descending
    assert np.abs(V.conj().T @ V - np.eye(n)).max() <= 1e-13           # unitary
    assert np.linalg.norm(A @ V - V * lam) <= 1e-12 * np.linalg.norm(A)
    if n >= 5:
        # leading well-separated invariant subspace agrees with LAPACK's
        _, U = np.linalg.eigh(A)
        U = U[:, ::-1]
        k = 3
        assert np.linalg.norm(V[:, :k] @ V[:, :k].conj().T - U[:, :k] @ U[:, :k].conj().T) <= 1e-9


def test_jacobi_2x2_closed_form(oracle):
    a, b, al = 2.0, -1.0, 0.7 - 1.9j
    A = np.array([[a, al], [np.conj(al), b]])
    lam, V, _ = oracle.jacobi(A)
    r = np.sqrt(((a - b) / 2) ** 2 + abs(al) ** 2)
    assert np.allclose(lam, [(a + b) / 2 + r, (a + b) / 2 - r], rtol=1e-15, atol=1e-15)
    assert np.linalg.norm(A @ V - V * lam) < 1e-14


def test_jacobi_degenerate_inputs(oracle):
    lam, V, sweeps = oracle.jacobi(np.zeros((4, 4), dtype=complex))
    assert (lam == 0).all() and np.array_equal(V, np.eye(4)) and sweeps == 0
    lam, V, _ = oracle.jacobi(np.diag([1.0, 3.0, 2.0]).astype(complex))
    assert np.array_equal(lam, [3.0, 2.0, 1.0])
    assert np.array_equal(np.abs(V), np.eye(3)[:, [1, 2, 0]])
    # repeated eigenvalues: any orthonormal basis is right -> check residual only
    q, _ = np.linalg.qr(cn(np.random.default_rng(0), (6, 6)))
    A = (q * np.array([5, 5, 5, 1, 1, 0.0])) @ q.conj().T
    lam, V, _ = oracle.jacobi((A + A.conj().T) / 2)
    assert np.allclose(lam, [5, 5, 5, 1, 1, 0], atol=1e-13)
    assert np.linalg.norm(A @ V - V * lam) < 1e-13


def test_eigenvalues_are_squared_singular_values(oracle):
    # Eq. 3: all-ones window -> lambda_i = sigma_i(C)^2
    rng = np.random.default_rng(3)
    iq = (cn(rng, (12, 6, 10)) * np.logspace(0, -3, 12)[:, None, None]).astype(np.complex64)
    R = oracle.gram(iq, np.ones(10), np.ones(6))
    lam, V, _ = oracle.jacobi(R)
    sv = np.linalg.svd(casorati(iq), compute_uv=False)
    assert np.abs(lam - sv ** 2).max() <= 1e-13 * sv[0] ** 2
    # right singular vectors = eigenvectors (up to phase): compare rank-1 projectors of the top ones
    _, _, Vh = np.linalg.svd(casorati(iq), full_matrices=False)
    for i in range(4):
        v = Vh[i].conj()
        assert np.linalg.norm(np.outer(v, v.conj()) - np.outer(V[:, i], V[:, i].conj())) < 1e-8


def test_unitary_temporal_mixing_leaves_spectrum(oracle):
    rng = np.random.default_rng(4)
    iq = cn(rng, (8, 5, 7)).astype(np.complex64)
    Q, _ = np.linalg.qr(cn(rng, (8, 8)))
    Cm = casorati(iq)
    gz, gx = oracle.axis_windows(7, 1, 2.0, 0.0)[0], oracle.axis_windows(5, 1, 2.0, 0.0)[0]
    w2 = np.outer(gx, gz).reshape(-1) ** 2
    R1 = (Cm.conj().T * w2) @ Cm
    C2 = Cm @ Q
    R2 = (C2.conj().T * w2) @ C2
    assert np.abs(oracle.gram(iq, gz, gx) - R1).max() < 1e-12
    l1, _, _ = oracle.jacobi(R1)
    l2, _, _ = oracle.jacobi((R2 + R2.conj().T) / 2)
    assert np.abs(l1 - l2).max() <= 1e-12 * l1[0]


# ---------------------------------------------------------------- cut-off and weights
def test_energy_cutoff_bruteforce(oracle):
    # hand-made spectra, rule: smallest 1-based m with cumulative energy > frac * total
    assert oracle.cutoff_energy(np.array([90.0, 9.0, 0.9, 0.1]), 0.995) == 3      # 99.9 > 99.5
    assert oracle.cutoff_energy(np.array([90.0, 9.0, 0.9, 0.1]), 0.90) == 2       # 90 is not > 90
    assert oracle.cutoff_energy(np.array([90.0, 9.0, 0.9, 0.1]), 0.89) == 1
    assert oracle.cutoff_energy(np.array([1.0, 1.0, 1.0, 1.0]), 0.5) == 3         # 2 is not > 2
    assert oracle.cutoff_energy(np.array([1.0, 1.0, 1.0, 1.0]), 1.0) == 4         # never exceeds
    assert oracle.cutoff_energy(np.array([10.0, 1.0, -5.0]), 0.95) == 2           # negatives clamp to 0
    rng = np.random.default_rng(5)
    for _ in range(50):
        lam = np.sort(rng.random(9) ** 4)[::-1]
        frac = rng.uniform(0.3, 0.999)
        cum = [lam[:m].sum() for m in range(1, 10)]
        want = next((m + 1 for m in range(9) if cum[m] > frac * lam.sum()), 9)
        assert oracle.cutoff_energy(lam, frac) == want


def test_median_cutoff_pins(oracle):
    # method 3 (Eq. 7): T = scale * median eigenvalue, c = # eigenvalues above T
    lam = np.array([100.0, 40.0, 9.0, 3.0, 2.0, 1.0, 0.5])                         # odd: median = 3
    assert oracle.cutoff_median(lam, 1.0) == 3                                     # 100, 40, 9 > 3
    assert oracle.cutoff_median(lam, 3.0) == 2                                     # 9 is not > 9
    assert oracle.cutoff_median(lam, 2.9) == 3
    assert oracle.cutoff_median(lam, 50.0) == 0
    lam = np.array([8.0, 6.0, 4.0, 2.0])                                           # even: median = 5
    assert oracle.cutoff_median(lam, 1.0) == 2
    assert oracle.cutoff_median(lam, 1.2) == 1                                     # 6 is not > 6
    assert oracle.cutoff_median(np.ones(6), 1.0) == 0                              # flat spectrum: nothing above
    # against numpy's median (same even-count convention as MATLAB) on random descending spectra
    rng = np.random.default_rng(11)
    for n in (2, 3, 8, 33, 128):
        for _ in range(20):
            lam = np.sort(rng.random(n) ** 6)[::-1]
            beta = rng.uniform(0.5, 20.0)
            assert oracle.cutoff_median(lam, beta) == int((lam > beta * np.median(lam)).sum())
    # the worked value in the paper's Fig. 2a (scaling factor 1.43) belongs to the authors' data:
    # it cannot be reproduced here; a low-rank-plus-white-noise spectrum stands in:
    lam = np.concatenate([[1e6, 3e4, 2e3], np.linspace(1.3, 0.7, 47)])
    assert oracle.cutoff_median(lam, 1.43) == 3


def test_slope_cutoff_pins(oracle):
    # method 2 as printed: slope of the eigenvalue curve y(n) = lambda_n, here relative to
    # its first point (reading 18 of DESIGN.md); c = (first n whose drop y(n) - y(n+1) is below T) - 1.
    # hand count: lambda / lambda_1 = 1, .5, .2, .19, .18, .17 -> drops .5, .3, .01, .01, .01
    lam = np.array([100.0, 50.0, 20.0, 19.0, 18.0, 17.0])
    assert oracle.cutoff_slope(lam, 0.05) == 2         # n = 3 is the first flat step: 2 components go
    assert oracle.cutoff_slope(lam, 0.4) == 1          # 0.3 < 0.4: only the first step is steep
    assert oracle.cutoff_slope(lam, 0.6) == 0          # already the first drop (0.5) is "flat"
    assert oracle.cutoff_slope(lam, 0.005) == 5        # never below 0.005: only the last component stays
    # the strict "<": a threshold exactly on a drop that floating point represents exactly (0.5) keeps that step steep
    assert oracle.cutoff_slope(np.array([8.0, 4.0, 3.0]), 0.5) == 1
    # exactly arithmetic curve (constant slope -1/16 per index, exact in binary): flat iff the threshold exceeds it
    lam = 1.0 - np.arange(12) / 16.0
    assert oracle.cutoff_slope(lam, 0.0624) == 11
    assert oracle.cutoff_slope(lam, 0.0626) == 0
    # brute force from the definition on random descending spectra: numpy's first difference of the curve
    rng = np.random.default_rng(5)
    for n in (2, 3, 9, 40, 128):
        for _ in range(20):
            lam = np.sort(rng.random(n) ** 8 + 1e-9)[::-1]
            T = 10.0 ** rng.uniform(-6, -0.5)
            slope = np.diff(lam / lam[0])                 # y(n+1) - y(n) <= 0
            flat = np.nonzero(slope > -T)[0]              # slope above the (negative) threshold: flat
            want = int(flat[0]) if flat.size else n - 1   # 0-based index of the first flat step = (1-based n) - 1
            assert oracle.cutoff_slope(lam, T) == want
    # unit-free through the normalisation by lambda_1 (a power of two keeps the quotients bit-identical)
    lam = np.concatenate([[4e5, 2e4, 900.0], np.linspace(1.3, 0.7, 29)])
    assert oracle.cutoff_slope(lam, 1e-3) == oracle.cutoff_slope(2.0 ** -30 * lam, 1e-3) == 3
    # differs from the dB variant where the curve is steep in dB but already flat on the linear scale:
    # drops 0.95, 0.04775, ... of lambda_1 (only the first is above 0.1) against 13.0, 13.5, 28.4, 0.07 dB
    assert oracle.cutoff_slope(lam, 0.1) == 1 and oracle.cutoff_slope_db(lam, 1.0) == 3
    assert oracle.cutoff_slope(np.array([5.0]), 0.1) == 0
    assert oracle.cutoff_slope(np.zeros(4), 0.1) == 0
    assert oracle.cutoff_slope(np.ones(6), 0.1) == 0   # flat spectrum: nothing stands out
    assert oracle.cutoff_slope(np.array([1.0, 0.5, 0.0, -1e-3]), 0.1) == 2   # no floor on the linear curve: 0 -> -1e-3 is flat


def test_slope_db_variant_pins(oracle):
    # named variant: the same rule on y(n) = 10 log10(lambda_n).  hand count: drops 10, 10, 30, 0.458, 0.512, 0.580 dB
    lam = np.array([1e6, 1e5, 1e4, 10.0, 9.0, 8.0, 7.0])
    assert oracle.cutoff_slope_db(lam, 1.1) == 3       # n = 4 is the first flat step: 3 components go
    assert oracle.cutoff_slope_db(lam, 0.5) == 3       # 0.458 < 0.5 too
    assert oracle.cutoff_slope_db(lam, 0.4) == 6       # never below 0.4 dB: only the last component stays
    assert oracle.cutoff_slope_db(lam, 10.5) == 0      # already the first drop (10 dB) is "flat"
    assert oracle.cutoff_slope_db(lam, 9.99) == 3      # the two 10 dB steps and the 30 dB step are steeper: n = 4 again
    # exactly geometric curve, 3 dB per step: flat iff the threshold exceeds 3 dB
    lam = 10.0 ** (-0.3 * np.arange(12))
    assert oracle.cutoff_slope_db(lam, 2.9) == 11
    assert oracle.cutoff_slope_db(lam, 3.1) == 0
    rng = np.random.default_rng(5)
    for n in (2, 3, 9, 40, 128):
        for _ in range(20):
            lam = np.sort(rng.random(n) ** 8 + 1e-9)[::-1]
            T = rng.uniform(0.05, 6.0)
            drops = 10 * np.log10(lam[:-1]) - 10 * np.log10(lam[1:])
            flat = np.nonzero(drops < T)[0]
            want = int(flat[0]) if flat.size else n - 1
            assert oracle.cutoff_slope_db(lam, T) == want
    lam = np.concatenate([[4e5, 2e4, 900.0], np.linspace(1.3, 0.7, 29)])
    assert oracle.cutoff_slope_db(lam, 1.1) == oracle.cutoff_slope_db(3.7e-9 * lam, 1.1) == 3
    assert oracle.cutoff_slope_db(np.array([5.0]), 1.1) == 0
    assert oracle.cutoff_slope_db(np.zeros(4), 1.1) == 0
    assert oracle.cutoff_slope_db(np.ones(6), 1.1) == 0
    # eigenvalues at or below zero are floored at 1e-12 lambda_1 (-120 dB): the step onto the floor is steep
    assert oracle.cutoff_slope_db(np.array([1.0, 0.5, 0.0, -1e-3]), 1.1) == 2


def test_curvature_cutoff_pins(oracle):
    # method 1 (Eq. 6): a log-eigenvalue curve made of two straight lines has zero
    # second difference everywhere except at the kink, so the maximum curvature sits exactly there
    N = 40
    n = np.arange(1, N + 1)
    for k0 in (3, 5, 9, 17, 21):
        f = np.where(n <= k0, 6.0 - 0.5 * (n - 1), 6.0 - 0.5 * (k0 - 1) - 0.02 * (n - k0))
        for beta in (0.3, 1.0, 2.5):
            assert oracle.cutoff_curvature(10.0 ** f, beta) == k0
    # the units of the eigenvalues enter through the paper's normalisation by log10(lambda_1):
    # a straight log-curve has no curvature anywhere -> first candidate (n = 2) by the tie rule
    assert oracle.cutoff_curvature(10.0 ** (5.0 - 0.1 * n), 1.0) == 2
    # the floor at 1e-12 lambda_1 (our reading) bends a curve that falls below it
    f = 6.0 - 0.5 * (n - 1)
    assert oracle.cutoff_curvature(10.0 ** f, 1.0) == 25                          # 6 - 0.5 * 24 = -6 = log10(1e-12 * 1e6)
    # degenerate inputs
    assert oracle.cutoff_curvature(np.array([4.0, 2.0]), 1.0) == 0              # N < 3: no interior point
    assert oracle.cutoff_curvature(np.array([1.0, 0.5, 0.1, 0.01]), 1.0) == 0   # log10(lambda_1) = 0
    assert oracle.cutoff_curvature(np.zeros(5), 1.0) == 0
    # a circle: y(n) on an arc of radius r has curvature 1/r everywhere; bending the arc more sharply
    # around one index must move the maximum there (numerical check of |y''|/(1+y'^2)^(3/2))
    N = 64
    n = np.arange(1, N + 1, dtype=np.float64)
    y = 40.0 - 0.05 * n - 3.0 / (1.0 + np.exp(-(n - 20.0) * 2.0))
    # logistic step centred at 20: |y''| peaks one to two samples either side of the centre, y' is largest at it
    lam = 10.0 ** (y * (6.0 / y[0]))                # y(1) -> log10(lambda_1) = 6; normalised curve = N * y / y[0] * beta
    k = oracle.cutoff_curvature(lam, 1.0)
    yy = 1.0 * N * np.log10(lam) / np.log10(lam[0])
    d1 = (yy[2:] - yy[:-2]) / 2; d2 = yy[2:] - 2 * yy[1:-1] + yy[:-2]
    assert k == int(np.argmax(np.abs(d2) / (1 + d1 ** 2) ** 1.5)) + 2 and 17 <= k <= 23


def test_adaptive_weights_pins(oracle):
    # method 6 (Eq. 10): wt_i = win(i) / lambda_i^beta, normalised to max 1
    from scipy.signal.windows import gaussian
    for N in (5, 32, 101):
        # flat spectrum (or beta -> 0): the weights are the window itself = right half of gausswin(2N-1, 2.5),
        # whose standard deviation in samples is (L-1)/(2 alpha) = (N-1)/2.5
        win = gaussian(2 * N - 1, std=(N - 1) / 2.5)[N - 1:]
        assert np.allclose(oracle.weights_adaptive(np.full(N, 7.0), 1.3), win, rtol=0, atol=1e-15)
        assert np.allclose(oracle.weights_adaptive(np.sort(np.random.default_rng(N).random(N))[::-1] + 1, 1e-12), win, atol=1e-10)
    # hand-computed: N = 3, lambda = (100, 10, 1), beta = 1: raw = [1/100, e^-0.78125/10, e^-3.125/1]
    raw = np.array([0.01, np.exp(-0.78125) / 10, np.exp(-3.125)])
    assert np.allclose(oracle.weights_adaptive(np.array([100.0, 10.0, 1.0]), 1.0), raw / raw.max(), rtol=1e-14)
    # scale invariance (normalisation removes lambda units), maximum exactly 1, floor at 1e-12 lambda_1
    lam = np.sort(np.random.default_rng(3).random(20) ** 5)[::-1] + 1e-3
    w = oracle.weights_adaptive(lam, 0.8)
    assert w.max() == 1.0 and (w >= 0).all()
    assert np.allclose(oracle.weights_adaptive(1e6 * lam, 0.8), w, rtol=1e-12)
    a = oracle.weights_adaptive(np.array([1.0, 0.5, 0.0, -1e-9]), 1.0)
    b = oracle.weights_adaptive(np.array([1.0, 0.5, 1e-12, 1e-12]), 1.0)
    assert np.array_equal(a, b)


def test_median_mode_runs_like_fixed_cut(oracle):
    # a window whose median rule gives c must equal the fixed-cut result with k_fixed = c
    iq = synth.random_cube(16, 12, 10, seed=4)
    gz = oracle.axis_windows(16, 1, 0.0, 0.0)[0]; gx = oracle.axis_windows(12, 1, 0.0, 0.0)[0]
    a = oracle.window(iq, gz, gx, synth.HARD_MEDIAN, cut_scale=1.5)
    b = oracle.window(iq, gz, gx, synth.HARD_FIXED, k_fixed=a["c"])
    assert a["c"] == int((a["lam"] > 1.5 * np.median(a["lam"])).sum())
    assert np.array_equal(a["wt"], b["wt"]) and np.array_equal(a["PDk"], b["PDk"])
    s1 = oracle.window(iq, gz, gx, synth.SOFT_MEDIAN, beta=0.7, cut_scale=1.5)
    s2 = oracle.window(iq, gz, gx, synth.SOFT_FIXED, k_fixed=a["c"], beta=0.7)
    assert np.array_equal(s1["wt"], s2["wt"])


def test_weights_closed_forms(oracle):
    assert np.array_equal(oracle.weights(6, False, 2, 0.5), [0, 0, 1, 1, 1, 1])
    assert np.array_equal(oracle.weights(3, False, 0, 0.5), [1, 1, 1])
    assert np.array_equal(oracle.weights(3, False, 3, 0.5), [0, 0, 0])
    wt = oracle.weights(8, True, 3, np.log(3.0))                                      # Eq. 9
    assert np.isclose(wt[2], 0.5, rtol=1e-15)            # i = k  -> 1/2
    assert np.isclose(wt[3], 0.75, rtol=1e-15)           # i = k+1, e^-beta = 1/3 -> 3/4
    assert np.isclose(wt[1], 0.25, rtol=1e-15)           # i = k-1 -> 1/4
    assert np.isclose(wt[4], 0.9, rtol=1e-15)            # i = k+2, e^-2beta = 1/9 -> 9/10
    assert (np.diff(wt) > 0).all()
    assert np.allclose(wt[:5] + wt[:5][::-1], 1.0)     # sigmoid is odd about i = k
    # beta -> infinity reproduces the hard weights except wt_k = 1/2
    big = oracle.weights(6, True, 2, 1e3)
    assert np.allclose(big, [0, 0.5, 1, 1, 1, 1], atol=1e-300)


# ---------------------------------------------------------------- filter matrix (Eqs. 4, 5)
def test_filter_projector_properties(oracle):
    rng = np.random.default_rng(6)
    n, c = 10, 3
    A, _, _ = rand_herm(rng, n, 1e4)
    lam, V, _ = oracle.jacobi((A + A.conj().T) / 2)
    F = oracle.filter_matrix(V, oracle.weights(n, False, c, 0.5))
    assert np.abs(F - F.conj().T).max() < 1e-14                       # Hermitian
    assert np.abs(F @ F - F).max() < 1e-13                            # idempotent
    assert np.isclose(np.trace(F).real, n - c, atol=1e-12)            # rank N - c
    Pi_c = V[:, :c] @ V[:, :c].conj().T
    assert np.abs(F - (np.eye(n) - Pi_c)).max() < 1e-13               # Eq. 4 == Eq. 5
    # against LAPACK's invariant subspace: F kills the c dominant eigenvectors of A
    _, U = np.linalg.eigh(A)
    assert np.abs(U[:, -c:].conj().T @ F).max() < 1e-9
    assert np.abs(oracle.filter_matrix(V, np.ones(n)) - np.eye(n)).max() < 1e-13      # keep all -> I
    wt = rng.random(n)
    assert np.abs(oracle.filter_matrix(V, wt) - (V * wt) @ V.conj().T).max() < 1e-14


# ---------------------------------------------------------------- projection + PD
def test_projection_allpass_and_trace_identity(oracle):
    rng = np.random.default_rng(7)
    N, Nx, Nz = 6, 8, 9
    iq = cn(rng, (N, Nx, Nz)).astype(np.complex64)
    gz, gx = oracle.axis_windows(Nz, 2, 3.0, 1.5)[1], oracle.axis_windows(Nx, 2, 2.5, 0.0)[0]
    w2 = np.outer(gx, gz) ** 2
    energy = (np.abs(iq.astype(np.complex128)) ** 2).sum(0)             # [Nx][Nz]
    PD = oracle.project_pd(iq, gz, gx, np.eye(N, dtype=complex))
    assert np.allclose(PD, w2 * energy, rtol=1e-13, atol=0)             # all components kept
    assert (PD[w2 == 0] == 0).all() and (w2 == 0).any()
    R = oracle.gram(iq, gz, gx)
    lam, V, _ = oracle.jacobi(R)
    for soft, c in [(False, 2), (True, 3)]:
        wt = oracle.weights(N, soft, c, 0.8)
        PD = oracle.project_pd(iq, gz, gx, oracle.filter_matrix(V, wt))
        # sum_p PD_k(p) = trace(F^H R F) = sum_i wt_i^2 lambda_i
        assert np.isclose(PD.sum(), (wt ** 2 * lam).sum(), rtol=1e-12)


def test_rank_r_clutter_is_removed(oracle):
    # exact rank-r clutter, zero blood: removing r components leaves round-off.  Fails if the Gram
    # and the projection disagree on which operand is conjugated (R-bar has conjugate eigenvectors).
    r, N = 3, 8
    iq = synth.rank_r_clutter(10, 7, N, r, seed=11)
    gz, gx = oracle.axis_windows(10, 1, 4.0, 0.0)[0], oracle.axis_windows(7, 1, 3.0, 0.0)[0]
    res = oracle.window(iq, gz, gx, oracle.HARD_FIXED, k_fixed=r)
    total = oracle.project_pd(iq, gz, gx, np.eye(N, dtype=complex)).sum()
    # complex64 storage of S = A B^H leaves a rank-deficiency error of ~1e-7 relative amplitude
    assert res["PDk"].sum() <= 1e-12 * total
    res2 = oracle.window(iq, gz, gx, oracle.HARD_FIXED, k_fixed=r - 1)
    assert res2["PDk"].sum() > 1e-4 * total                     # one clutter component left


def test_dc_removal_textbook_case(oracle):
    # constant-in-time tissue on half the pixels, a pure slow-time tone (integer cycles, so orthogonal
    # to DC) on the other half: R = |T|^2 11^H + |b|^2 u u^H exactly, v1 = 1/sqrt(N), and removing c = 1
    # component is the classical DC-removal (mean-subtraction) clutter filter.
    rng = np.random.default_rng(8)
    N, Nx, Nz = 16, 6, 6
    tissue = cn(rng, (1, Nx, Nz)) * 100.0
    tissue[:, :, 3:] = 0
    blood = cn(rng, (1, Nx, Nz))
    blood[:, :, :3] = 0
    tone = np.exp(2j * np.pi * 3 * np.arange(N) / N)[:, None, None]
    iq = (tissue + blood * tone).astype(np.complex64)
    res = oracle.window(iq, np.ones(Nz), np.ones(Nx), oracle.HARD_FIXED, k_fixed=1)
    s = iq.astype(np.complex128)
    ref = (np.abs(s - s.mean(0, keepdims=True)) ** 2).sum(0)
    assert np.allclose(res["PDk"], ref, rtol=1e-5, atol=1e-9 * ref.max())
    assert np.allclose(res["PDk"][:, 3:], N * np.abs(blood[0, :, 3:]) ** 2, rtol=1e-5)
    assert np.allclose(np.abs(res["V"][:, 0]), 1 / np.sqrt(N), rtol=1e-6)


def _bruteforce_window(iq, w, soft, c, beta):
    """The paper's own data flow, literally: C_w = W C (Eq. 11), R = C_w^H C_w (Eq. 12), EVD (Eq. 2,
    LAPACK), C^ = C_w V L^ V^H (Eq. 4), PD = sum_t |C^|^2."""
    Cm = casorati(iq)
    Cw = w.reshape(-1, 1) * Cm
    R = Cw.conj().T @ Cw
    lam, V = np.linalg.eigh(R)
    lam, V = lam[::-1], V[:, ::-1]
    i = np.arange(1, len(lam) + 1)
    wt = 1 / (1 + np.exp(-beta * (i - c))) if soft else (i > c).astype(float)
    Chat = Cw @ (V * wt) @ V.conj().T
    return (np.abs(Chat) ** 2).sum(1).reshape(iq.shape[1:]), lam


def test_bruteforce_tiny_localized(oracle):
    # 3 x 2 px, N = 3, K = 2 windows (and a slightly larger case), whole path vs the literal version
    for (Nz, Nx, N, Kz, Kx, sg, tr, soft, c, seed) in [(3, 2, 3, 2, 1, 1.0, 0.0, False, 1, 0),
                                                        (6, 5, 4, 2, 2, 2.0, 1.2, True, 2, 1),
                                                        (6, 5, 4, 2, 2, 2.0, 1.2, False, 2, 2)]:
        iq = synth.random_cube(Nz, Nx, N, seed)
        iq = (iq * np.array([30.0, 5.0, 1.0, 0.2])[:N, None, None]).astype(np.complex64)
        mode = oracle.SOFT_FIXED if soft else oracle.HARD_FIXED
        out = oracle.run(iq, Kz, Kx, sg, sg, tr, mode, k_fixed=c, beta=0.7)
        gz, gx = oracle.axis_windows(Nz, Kz, sg, tr), oracle.axis_windows(Nx, Kx, sg, tr)
        PD = np.zeros((Nx, Nz))
        for kx in range(Kx):
            for kz in range(Kz):
                pdk, lam = _bruteforce_window(iq, np.outer(gx[kx], gz[kz]), soft, c, 0.7)
                assert np.allclose(out["lam"][kx * Kz + kz], lam, rtol=0, atol=1e-12 * lam[0])
                PD += pdk / pdk.mean()
        assert np.allclose(out["PD"], PD, rtol=1e-9)


# ---------------------------------------------------------------- combination (Eq. 13)
def test_combine_properties(oracle):
    rng = np.random.default_rng(9)
    pk = rng.random((4, 5, 6))
    pk[2] = 0.0                                            # a window with zero flow power -> alpha = 0
    PD, alpha = oracle.combine(pk)
    assert alpha[2] == 0.0
    assert np.allclose(alpha[[0, 1, 3]], 1.0 / pk[[0, 1, 3]].mean(axis=(1, 2)))
    assert np.isclose(PD.sum(), 30 * 3)                    # each alpha_k PD_k has unit mean
    PD2, _ = oracle.combine(pk * np.array([3.0, 0.1, 7.0, 100.0])[:, None, None])
    assert np.allclose(PD, PD2)                            # per-window amplitude scaling cancels
    PD3, _ = oracle.combine(np.stack([pk[0]] * 3))
    assert np.allclose(PD3, 3 * pk[0] / pk[0].mean())      # K identical windows -> K x single


def test_run_invariances_and_composition(oracle):
    cfg = synth.scaled_config(synth.baseline_configs()[0], Nz=24, Nx=20, N=8, n_frames=8)
    iq = synth.generate(cfg)
    f = cfg.filt
    a = oracle.run(iq, 2, 2, 6.0, 5.0, 2.0, oracle.SOFT_ENERGY, frac=0.9, beta=0.5)
    b = oracle.run((iq * (0.3 - 2.0j)).astype(np.complex64), 2, 2, 6.0, 5.0, 2.0, oracle.SOFT_ENERGY, frac=0.9, beta=0.5)
    assert np.allclose(a["PD"], b["PD"], rtol=1e-5)                  # S -> cS leaves PD_final unchanged
    assert np.isclose(a["PD"].sum(), 4 * iq.shape[1] * iq.shape[2], rtol=1e-12)
    # run() == per-step functions composed by hand
    gz, gx = oracle.axis_windows(24, 2, 6.0, 2.0), oracle.axis_windows(20, 2, 5.0, 2.0)
    pks = []
    for kx in range(2):
        for kz in range(2):
            R = oracle.gram(iq, gz[kz], gx[kx])
            lam, V, _ = oracle.jacobi(R)
            c = oracle.cutoff_energy(lam, 0.9)
            assert c == a["c"][kx * 2 + kz]
            F = oracle.filter_matrix(V, oracle.weights(8, True, c, 0.5))
            pks.append(oracle.project_pd(iq, gz[kz], gx[kx], F))
    PD, _ = oracle.combine(np.stack(pks))
    assert np.allclose(PD, a["PD"], rtol=1e-12)
    # the optional V output of run(): the eigenvectors of each window, descending order (what the GPU
    # parity tests gate every window's clutter projector against), pinned to LAPACK on the same R
    v = oracle.run(iq, 2, 2, 6.0, 5.0, 2.0, oracle.SOFT_ENERGY, frac=0.9, beta=0.5, want_R=True, want_V=True)
    assert np.array_equal(v["PD"], a["PD"]) and np.array_equal(v["lam"], a["lam"])
    for k in range(4):
        R, V, lam = v["R"][k], v["V"][k], v["lam"][k]
        assert np.allclose(V.conj().T @ V, np.eye(8), atol=1e-13)
        assert np.linalg.norm(R @ V - V * lam) <= 1e-12 * np.linalg.norm(R)
        wl, Vl = np.linalg.eigh(R)
        c = int(v["c"][k])
        Pl = Vl[:, ::-1][:, :c] @ Vl[:, ::-1][:, :c].conj().T
        assert np.linalg.norm(V[:, :c] @ V[:, :c].conj().T - Pl) <= 1e-10


# ---------------------------------------------------------------- method 4: spatial NCC cut-off (Eq. 8)
def test_left_singular_vectors_pins(oracle):
    # C V = U D, lambda_i = sigma_i^2.  The magnitudes |u_i(p)| must be those of LAPACK's left
    # singular vectors of the (windowed) Casorati matrix; each u_i has unit norm.
    rng = np.random.default_rng(21)
    Nz, Nx, N = 7, 5, 6
    iq = (cn(rng, (N, Nx, Nz)) * np.array([9.0, 4.0, 2.0, 1.0, 0.5, 0.2])[:, None, None]).astype(np.complex64)
    for gz, gx in ((np.ones(Nz), np.ones(Nx)), (np.linspace(0.2, 1.0, Nz), np.array([1.0, 0.5, 0.0, 0.7, 0.9]))):
        R = oracle.gram(iq, gz, gx)
        lam, V, _ = oracle.jacobi(R)
        Um = oracle.left_singular_mag(iq, gz, gx, lam, V)                     # [Nx][Nz][N]
        Cw = np.outer(gx, gz).reshape(-1, 1) * casorati(iq)
        U, S, Vh = np.linalg.svd(Cw, full_matrices=False)
        assert np.allclose(S ** 2, lam, rtol=1e-10)
        assert np.allclose(Um.reshape(-1, N), np.abs(U), rtol=0, atol=1e-9)
        assert np.allclose((Um.reshape(-1, N) ** 2).sum(0), 1.0, rtol=1e-10)
        assert (Um[gx == 0] == 0).all()                                       # outside the window support
    # a component with lambda = 0 (rank-deficient data) has no left singular vector: |u| = 0 by our reading
    iq2 = synth.rank_r_clutter(6, 5, 5, 2, seed=3)
    R = oracle.gram(iq2, np.ones(6), np.ones(5))
    lam, V, _ = oracle.jacobi(R)
    Um = oracle.left_singular_mag(iq2, np.ones(6), np.ones(5), lam, V)
    assert (Um[..., 2:] == 0).all() and np.allclose((Um[..., :2] ** 2).sum((0, 1)), 1.0, rtol=1e-6)


def test_ncc_cutoff_pins(oracle):
    # Eq. 8 with the simplified images of PAPER.md:107 (fn components on either side of k).
    # hand-built: components 1..k0 live on pixels [0, 10), components k0+1.. on pixels [10, 20): at k = k0 the tissue
    # and blood images have disjoint supports -> NCC = 0 exactly; every other k mixes the two sets on one side.
    P, N, fn = 20, 12, 5
    for k0 in (3, 5, 6):
        U = np.zeros((P, N))
        U[:10, :k0] = 1.0 + 0.1 * np.arange(k0)
        U[10:, k0:] = 2.0 + 0.1 * np.arange(N - k0)
        k, ncc = oracle.cutoff_ncc(U, fn)
        assert k == k0 and ncc[k0 - 1] == 0.0 and (np.delete(ncc, k0 - 1) > 0).all() and np.isinf(ncc[-1])
    # identical spatial patterns in every component: NCC = 1 everywhere, the lowest k wins the tie
    U = np.tile(np.linspace(1.0, 2.0, P)[:, None], (1, N))
    k, ncc = oracle.cutoff_ncc(U, fn)
    assert k == 1 and np.allclose(ncc[:-1], 1.0, rtol=1e-14)
    # a k whose tissue (or blood) image vanishes everywhere is never chosen
    U = np.abs(np.random.default_rng(0).standard_normal((P, N)))
    U[:, :2] = 0.0
    k, ncc = oracle.cutoff_ncc(U, 2)                                           # I_T(1), I_T(2) = 0
    assert np.isinf(ncc[0]) and np.isinf(ncc[1]) and k >= 3
    # brute force from the definition in numpy (1-based sums clipped to 1..N), random magnitudes, several fn
    rng = np.random.default_rng(8)
    for n, f in ((4, 5), (9, 2), (16, 5), (33, 5), (33, 1)):
        U = np.abs(rng.standard_normal((37, n))) ** 3
        k, ncc = oracle.cutoff_ncc(U, f)
        ref = np.full(n, np.inf)
        for kk in range(1, n):
            it = U[:, max(kk - f, 0):kk].sum(1)                                 # i = kk-f+1 .. kk  (0-based columns kk-f .. kk-1)
            ib = U[:, kk:min(kk + f, n)].sum(1)                                 # i = kk+1 .. kk+f
            ref[kk - 1] = (it * ib).sum() / np.sqrt((it * it).sum() * (ib * ib).sum())
        assert np.allclose(ncc, ref, rtol=1e-12) and k == int(np.argmin(ref)) + 1
    # NCC is invariant to a common scaling of all magnitudes and to a permutation of the pixels
    U = np.abs(rng.standard_normal((50, 14)))
    k1, n1 = oracle.cutoff_ncc(U, 5)
    k2, n2 = oracle.cutoff_ncc(7.3 * U[rng.permutation(50)], 5)
    assert k1 == k2 and np.allclose(n1, n2, rtol=1e-12)


def test_ncc_mode_runs_like_fixed_cut(oracle):
    # method 4 end to end: the window's cut-off is the NCC minimum of its own left singular vectors, and
    # the image equals the fixed-cut image with that k (hard, and method 5's sigmoid around it)
    cfg = synth.scaled_config(synth.baseline_configs()[0], Nz=24, Nx=20, N=16, n_frames=16)
    iq = synth.generate(cfg)
    for mode_ncc, mode_fix in ((oracle.HARD_NCC, oracle.HARD_FIXED), (oracle.SOFT_NCC, oracle.SOFT_FIXED)):
        a = oracle.run(iq, 2, 1, 8.0, 8.0, 3.0, mode_ncc, beta=0.7, want_R=True)
        gz, gx = oracle.axis_windows(24, 2, 8.0, 3.0), oracle.axis_windows(20, 1, 8.0, 3.0)
        PD = np.zeros((20, 24))
        for kz in range(2):
            lam, V, _ = oracle.jacobi(a["R"][kz])
            k, _ = oracle.cutoff_ncc(oracle.left_singular_mag(iq, gz[kz], gx[0], lam, V), 5)
            assert k == a["c"][kz] and 1 <= k <= 15
            w = oracle.window(iq, gz[kz], gx[0], mode_fix, k_fixed=k, beta=0.7)
            PD += w["PDk"] / w["mean"]
        assert np.allclose(a["PD"], PD, rtol=1e-12)


def test_top_modes_are_the_hard_modes_on_the_oracle_side(oracle):
    """LCF_HARD_FIXED_TOP / LCF_HARD_ENERGY_TOP name a way of computing (leading eigenpairs only, include/lcf.h), not
    another filter: the oracle's answer for them is its answer for LCF_HARD_FIXED / LCF_HARD_ENERGY, from the full
    decomposition (Eq. 4).  Pinned independently of the mode plumbing: the image of a hard cut is the
    slow-time power of (I - Pi_c) applied to the windowed data, Pi_c from numpy.linalg.eigh of the oracle's own R."""
    cfg = synth.scaled_config(synth.baseline_configs()[0], Nz=24, Nx=20, N=16, n_frames=16)
    iq = synth.generate(cfg)
    for top, base, k in ((oracle.HARD_FIXED_TOP, oracle.HARD_FIXED, 3), (oracle.HARD_ENERGY_TOP, oracle.HARD_ENERGY, 0)):
        a = oracle.run(iq, 2, 1, 8.0, 8.0, 3.0, top, k_fixed=k, frac=0.99, want_R=True, want_F=True)
        b = oracle.run(iq, 2, 1, 8.0, 8.0, 3.0, base, k_fixed=k, frac=0.99, want_F=True)
        assert np.array_equal(a["c"], b["c"]) and np.array_equal(a["PD"], b["PD"]) and np.array_equal(a["F"], b["F"])
        for kz in range(2):
            lam, U = np.linalg.eigh(a["R"][kz])
            lam, U = lam[::-1], U[:, ::-1]
            c = int(a["c"][kz])
            if top == oracle.HARD_ENERGY_TOP:
                assert c == int(np.searchsorted(np.cumsum(lam), 0.99 * lam.sum(), side="right") + 1)
            F = np.eye(16) - U[:, :c] @ U[:, :c].conj().T
            assert np.abs(a["F"][kz] - F).max() <= 1e-10


def test_fig2f_sigmoid_example(oracle):
    """The paper's one stated example of Eq. 9 (Fig. 2f: beta = 2, k = 13) against the logistic table values
    in tests/golden/fig2f_sigmoid_beta2_k13.txt."""
    from pathlib import Path
    rows = [l.split() for l in (Path(__file__).parent / "golden" / "fig2f_sigmoid_beta2_k13.txt").read_text().splitlines()
            if l.strip() and not l.startswith("#")]
    wt = oracle.weights(50, True, 13, 2.0)
    assert len(rows) == 7
    for i, v in rows:
        assert np.isclose(wt[int(i) - 1], float(v), rtol=1e-14), (i, wt[int(i) - 1], v)
