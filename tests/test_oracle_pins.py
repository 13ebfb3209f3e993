"""Pins of the fp64 oracle against things other than itself (SURVEY.md §8(c) "What pins each part").

CPU only.  numpy FFTs / dense linear algebra appear HERE (tests) as independent library cross-checks,
never inside the oracle.
"""
from pathlib import Path

import numpy as np
import pytest

import oracle

GOLD = Path(__file__).parent / "golden"
rng = np.random.default_rng(20210604)


def T(x):
    """(T f)[j] = f[(nt-j) % nt] along the last axis."""
    return np.roll(x[..., ::-1], 1, axis=-1)


# ---------------------------------------------------------------- band, weights, projector (O1, O2)
def test_band_matches_baseline_json():
    # BASELINE.json configs: "about 451 bins" for 5-60 Hz at nt*dt = 8.192 s; 41..491 / 11..122
    assert oracle.band(2048, 0.004, 5.0, 60.0) == (41, 491, 451)
    assert oracle.band(4096, 0.002, 5.0, 60.0) == (41, 491, 451)
    assert oracle.band(512, 0.004, 5.0, 60.0) == (11, 122, 112)
    assert oracle.band(32, 1.0, 0.0, 0.5) == (0, 16, 17)          # all-pass includes DC and Nyquist
    assert oracle.band(512, 0.004, 0.0, 125.0) == (0, 256, 257)   # Nyquist edge despite rounding of 1/(nt dt)


def test_trapezoid_weights():
    np.testing.assert_array_equal(oracle.weights(5, 10.0), [5.0, 10.0, 10.0, 10.0, 5.0])
    np.testing.assert_array_equal(oracle.weights(1, 3.0), [3.0])
    # integrates a linear function exactly
    x = np.arange(7) * 2.5
    assert abs(np.dot(oracle.weights(7, 2.5), 3 * x + 1) - (1.5 * 15.0 ** 2 + 15.0)) < 1e-12


@pytest.mark.parametrize("nt,klo,khi", [(64, 3, 17), (64, 0, 32), (128, 0, 5), (32, 7, 16)])
def test_band_kernel_is_the_projector(nt, klo, khi):
    b = oracle.band_kernel(nt, klo, khi)
    # equals the inverse DFT of the 0/1 band mask (library cross-check)
    mask = np.zeros(nt // 2 + 1)
    mask[klo:khi + 1] = 1.0
    np.testing.assert_allclose(b, np.fft.irfft(mask, nt), atol=1e-15)
    # idempotent: b (*) b = b
    np.testing.assert_allclose(oracle.apply_band(b, b), b, atol=1e-14)
    # sum_q b[q] = [0 in B]
    assert abs(b.sum() - (1.0 if klo == 0 else 0.0)) < 1e-13
    # in-band cosine passes unchanged, out-of-band one is annihilated
    j = np.arange(nt)
    kin = (klo + khi) // 2
    x = np.cos(2 * np.pi * kin * j / nt + 0.3)
    np.testing.assert_allclose(oracle.apply_band(b, x), x, atol=1e-13)
    kout = khi + 1 if khi < nt // 2 else klo - 1
    if 0 <= kout <= nt // 2:
        y = oracle.apply_band(b, np.cos(2 * np.pi * kout * j / nt + 0.3))
        assert np.abs(y).max() < 1e-13
    # Parseval against a naive O(nt^2) DFT
    x = rng.standard_normal(nt)
    W = np.exp(-2j * np.pi * np.outer(np.arange(nt // 2 + 1), j) / nt)
    X = W @ x
    c = np.full(nt // 2 + 1, 2.0)
    c[0] = 1.0
    c[nt // 2] = 1.0
    lhs = np.sum(oracle.apply_band(b, x) ** 2)
    rhs = np.sum((c * np.abs(X) ** 2)[klo:khi + 1]) / nt
    assert abs(lhs - rhs) < 1e-11 * max(1.0, rhs)


# ---------------------------------------------------------------- window (O3)
def test_window_table_and_support():
    nt, dt, eps = 64, 0.004, 8
    td = np.array([0.0, 0.0339, 0.0341, 0.05, 0.1, 0.2, 1.0], dtype=np.float32)
    h = oracle.window(td, nt, dt, eps)
    m = np.floor(td.astype(np.float64) / dt + 0.5)
    np.testing.assert_array_equal(h, np.clip(m - eps, 0, nt // 2).astype(np.int32))
    assert h[0] == 0 and h[-1] == nt // 2
    for hv in [0, 1, 2, 5, nt // 2 - 1, nt // 2]:
        th = oracle.theta(nt, hv)
        assert th.sum() == max(2 * hv - 1, 0)          # kept samples per trace
        np.testing.assert_array_equal(th, T(th))       # symmetric in +-t  => Theta T = T Theta
        js = np.where(np.arange(nt) < nt // 2, np.arange(nt), np.arange(nt) - nt)
        np.testing.assert_array_equal(th, (np.abs(js) < hv).astype(float))


# ---------------------------------------------------------------- synthesis operator (O5a)
def test_delta_spike_R_is_an_exact_circular_shift():
    # R[s][r][j] = delta_sr delta_{j,q} / (w[s] dt), all-pass band  =>  (R N) = N shifted by q, exactly.
    n, nt, nfoc, dt, dx = 5, 32, 3, 0.5, 2.0
    w = oracle.weights(n, dx)
    klo, khi, _ = oracle.band(nt, dt, 0.0, 1.0 / (2 * dt))
    assert (klo, khi) == (0, nt // 2)
    for q in (0, 1, 7, 31):
        R = np.zeros((n, n, nt), dtype=np.float32)
        for s in range(n):
            R[s, s, q] = 1.0 / (w[s] * dt)               # 1 or 2: exact in fp32
        N = rng.standard_normal((nfoc, n, nt))
        S = oracle.synthesis(R, N, dt, w, klo, khi)
        np.testing.assert_allclose(S, np.roll(N, q, axis=-1), atol=2e-14)


def _rand_problem(n=6, nt=32, nfoc=2, nrout=None):
    nrout = n if nrout is None else nrout
    R = rng.standard_normal((n, nrout, nt)).astype(np.float32)
    N = rng.standard_normal((nfoc, n, nt))
    return R, N


def test_linearity_in_R_and_N():
    n, nt, dt, dx = 6, 32, 0.004, 10.0
    w = oracle.weights(n, dx)
    klo, khi, _ = oracle.band(nt, dt, 20.0, 90.0)
    R1, N1 = _rand_problem()
    R2, N2 = _rand_problem()
    a, c = 2.0, -0.5      # exact scalings in fp32
    lhs = oracle.synthesis((a * R1 + c * R2).astype(np.float32), N1, dt, w, klo, khi)
    rhs = a * oracle.synthesis(R1, N1, dt, w, klo, khi) + c * oracle.synthesis(R2, N1, dt, w, klo, khi)
    Rsum = (a * R1 + c * R2).astype(np.float32)
    # fp32 rounding of the summed R is the only inexactness
    err_in = np.abs(Rsum.astype(np.float64) - (a * R1.astype(np.float64) + c * R2.astype(np.float64))).max()
    assert np.abs(lhs - rhs).max() < 1e-13 + 1e3 * err_in
    lhs = oracle.synthesis(R1, 0.7 * N1 - 1.3 * N2, dt, w, klo, khi)
    rhs = 0.7 * oracle.synthesis(R1, N1, dt, w, klo, khi) - 1.3 * oracle.synthesis(R1, N2, dt, w, klo, khi)
    np.testing.assert_allclose(lhs, rhs, atol=1e-13 * np.abs(rhs).max())


def _synthesis_fft(R, N, dt, w, klo, khi):
    """Textbook identity: circular convolution = irfft(rfft * rfft); integrates over the SHOT index (G10)."""
    nt = R.shape[-1]
    Rf = np.fft.rfft(R.astype(np.float64), axis=-1)           # [s][r][k]
    Nf = np.fft.rfft(N, axis=-1)                               # [f][s][k]
    Sf = dt * np.einsum("s,srk,fsk->frk", w, Rf, Nf)
    mask = np.zeros(nt // 2 + 1)
    mask[klo:khi + 1] = 1.0
    return np.fft.irfft(Sf * mask, nt, axis=-1)


@pytest.mark.parametrize("n,nrout,nt,nfoc,band", [(6, 6, 32, 2, (20.0, 90.0)), (7, 3, 64, 3, (0.0, 125.0)),
                                                   (1, 1, 16, 1, (30.0, 60.0))])
def test_matches_fft_identity_nonsymmetric_R(n, nrout, nt, nfoc, band):
    dt, dx = 0.004, 10.0
    w = oracle.weights(n, dx)
    klo, khi, _ = oracle.band(nt, dt, *band)
    R, N = _rand_problem(n, nt, nfoc, nrout)                   # R[s][r] != R[r][s]: a transposed operand fails
    S = oracle.synthesis(R, N, dt, w, klo, khi)
    ref = _synthesis_fft(R, N, dt, w, klo, khi)
    np.testing.assert_allclose(S, ref, atol=1e-12 * np.abs(ref).max())


def test_zero_skipping_is_exact_with_sparse_inputs():
    n, nt, dt, dx = 5, 64, 0.004, 10.0
    w = oracle.weights(n, dx)
    klo, khi, _ = oracle.band(nt, dt, 10.0, 100.0)
    R, N = _rand_problem(n, nt, 2)
    R[:, :, nt // 2:] = 0.0
    R[1, 2, :] = 0.0
    N[:, :, 5:40] = 0.0
    N[1, 3, :] = 0.0
    ref = _synthesis_fft(R, N, dt, w, klo, khi)
    np.testing.assert_allclose(oracle.synthesis(R, N, dt, w, klo, khi), ref, atol=1e-12 * np.abs(ref).max())


# ---------------------------------------------------------------- signs, window polarity, G / G+ / G- (G1-G5)
def _goupillaud(rs, zF, nsteps):
    """Brute-force 1-D wavefield by time stepping (textbook Goupillaud medium; independent of the oracle).

    Unit downgoing impulse at depth 0 at t = 0, transparent surface.  Interface j (1-based) at depth 2j in
    one-way-time samples; flux-normalised scattering: +r from above, -r from below, sqrt(1-r^2) through.
    Returns R(t) = upgoing field at depth 0, and D(t), U(t) = down/upgoing fields at the (odd) depth zF."""
    L = len(rs)
    zmax = 2 * L + 2
    d = np.zeros(zmax + 1)
    u = np.zeros(zmax + 1)
    d[0] = 1.0
    R = np.zeros(nsteps)
    D = np.zeros(nsteps)
    U = np.zeros(nsteps)
    for t in range(nsteps):
        R[t], D[t], U[t] = u[0], d[zF], u[zF]
        for j in range(1, L + 1):
            z, r = 2 * j, rs[j - 1]
            tau = np.sqrt(1 - r * r)
            d[z], u[z] = tau * d[z] - r * u[z], r * d[z] + tau * u[z]
        d = np.concatenate(([0.0], d[:-1]))
        u = np.concatenate((u[1:], [0.0]))
    return R, D, U


@pytest.mark.parametrize("k", [0, 1, 2, 4])
def test_1d_layered_medium_exact_green_functions(k):
    rs = np.array([0.3, -0.25, 0.2, 0.28, -0.15])
    nt, Lr = 256, 100
    zF = 2 * k + 1                                           # focal point mid-layer k, t_d = 2k+1
    Rt, D, U = _goupillaud(rs, zF, nt)
    R = np.zeros((1, 1, nt), dtype=np.float32)
    R[0, 0, :Lr] = Rt[:Lr]
    Td = np.prod(np.sqrt(1 - rs[:k] ** 2))
    Gd = np.zeros((1, 1, nt), dtype=np.float32)
    Gd[0, 0, zF] = Td
    td = np.array([[zF]], dtype=np.float32)
    out = oracle.marchenko(R, Gd, td, dt=1.0, dx=1.0, fmin=0.0, fmax=0.5, niter=60, eps=0)
    Tm = Lr - zF - 1                                          # exact up to the truncation of R
    tol = 5e-7                                                # fp32 rounding of the inputs R, G_d
    assert np.abs(out["Gplus"][0, 0, :Tm] - Td ** 2 * D[:Tm]).max() < tol
    assert np.abs(out["Gminus"][0, 0, :Tm] - Td ** 2 * U[:Tm]).max() < tol
    assert np.abs(out["G"][0, 0, :Tm] - Td ** 2 * (D + U)[:Tm]).max() < tol
    for nm in ("G", "Gplus", "Gminus"):                       # causal: nothing at negative times
        assert np.abs(out[nm][0, 0, nt // 2 + 1:]).max() < 1e-12
    assert np.abs(D).max() > 0.5                              # the check is not vacuous


def test_golden_single_interface_closed_form():
    vals = {}
    for line in (GOLD / "single_interface_1d.txt").read_text().splitlines():
        if line.startswith("#") or not line.strip():
            continue
        p = line.split()
        vals[p[0]] = (float(p[1]),) if len(p) == 2 else (int(p[1]), float(p[2]))
    r, tau = vals["r"][0], vals["tau"][0]
    nt = 32
    R = np.zeros((1, 1, nt), dtype=np.float32)
    R[0, 0, 4] = r
    Gd = np.zeros((1, 1, nt), dtype=np.float32)
    Gd[0, 0, 3] = tau
    out = oracle.marchenko(R, Gd, np.array([[3.0]], np.float32), 1.0, 1.0, 0.0, 0.5, niter=6, eps=0)
    fields = {"f1plus": out["f1plus"], "f1min": out["f1min"], "N0": out["N_iters"][0], "Gplus": out["Gplus"],
              "G": out["G"]}
    for nm, arr in fields.items():
        t, v = vals[nm]
        exp = np.zeros(nt)
        exp[t % nt] = v
        np.testing.assert_allclose(arr[0, 0], exp, atol=1e-7, err_msg=nm)
    assert np.abs(out["Gminus"]).max() < 1e-7
    assert np.abs(out["N_iters"][1:]).max() < 1e-15   # all-pass kernel b = delta up to rounding


# ---------------------------------------------------------------- bookkeeping invariants (O5b, O5d, O6)
@pytest.mark.parametrize("niter", [1, 2, 5])
def test_accumulation_invariants(niter):
    n, nt, nfoc, dt, dx = 5, 32, 2, 0.004, 10.0
    R = (0.3 * rng.standard_normal((n, n, nt)) / (dt * dx * n)).astype(np.float32)
    Gd = rng.standard_normal((nfoc, n, nt)).astype(np.float32)
    td = (dt * rng.uniform(6, 14, size=(nfoc, n))).astype(np.float32)
    fmin, fmax, eps = 20.0, 100.0, 2
    o = oracle.marchenko(R, Gd, td, dt, dx, fmin, fmax, niter, eps)
    w = oracle.weights(n, dx)
    klo, khi, _ = oracle.band(nt, dt, fmin, fmax)
    syn = lambda x: oracle.synthesis(R, x, dt, w, klo, khi)
    Nlast = o["N_iters"][-1]
    scale = np.abs(o["f2"]).max()
    np.testing.assert_allclose(o["f2"], o["f1plus"] - T(o["f1min"]), atol=1e-13 * scale)
    np.testing.assert_allclose(o["pmin"], syn(o["f2"] - Nlast), atol=1e-12 * scale)
    np.testing.assert_allclose(o["G"] - (o["Gplus"] + o["Gminus"]), -syn(Nlast), atol=1e-12 * scale)
    # f2 is the plain sum of the iterates, and every iterate lives inside its window
    np.testing.assert_allclose(o["f2"], T(Gd.astype(np.float64)) + o["N_iters"].sum(axis=0), atol=1e-13 * scale)
    h = oracle.window(td, nt, dt, eps)
    for f in range(nfoc):
        for r in range(n):
            th = oracle.theta(nt, h[f, r])
            assert np.all(o["N_iters"][:, f, r, th == 0] == 0.0)
    # one Neumann step from the definition: N_0 = -Theta T R (T G_d)
    N0 = -np.stack([[oracle.theta(nt, h[f, r]) for r in range(n)] for f in range(nfoc)]) * T(syn(T(Gd.astype(np.float64))))
    np.testing.assert_allclose(o["N_iters"][0], N0, atol=1e-13 * scale)


# ---------------------------------------------------------------- the Neumann iteration as a whole
def test_geometric_series_closed_form_dense_matrices():
    """Sum_{k=0}^{K} A^k b = (I - A)^{-1} (I - A^{K+1}) b with A = -Theta T R built densely from the definition."""
    n, nt, dt, dx, eps, K = 4, 16, 0.004, 10.0, 1, 9
    fmin, fmax = 30.0, 110.0
    R = rng.standard_normal((n, n, nt)).astype(np.float32)
    td = (dt * rng.uniform(4, 8, size=(1, n))).astype(np.float32)
    w = oracle.weights(n, dx)
    klo, khi, _ = oracle.band(nt, dt, fmin, fmax)
    h = oracle.window(td, nt, dt, eps)[0]
    # dense operator from the definition, brute force: row (r, j), column (s, j')
    mask = np.zeros(nt // 2 + 1)
    mask[klo:khi + 1] = 1.0
    PB = np.array([np.fft.irfft(np.fft.rfft(e) * mask, nt) for e in np.eye(nt)]).T      # nt x nt projector
    Tm = np.zeros((nt, nt))
    for j in range(nt):
        Tm[j, (nt - j) % nt] = 1.0
    Tall = np.kron(np.eye(n), Tm)
    Th = np.diag(np.concatenate([oracle.theta(nt, h[r]) for r in range(n)]))

    def dense_A(Rx):
        Rop = np.zeros((n * nt, n * nt))
        for r in range(n):
            for s in range(n):
                Cm = np.array([[Rx[s, r, (j - jp) % nt] for jp in range(nt)] for j in range(nt)], dtype=np.float64)
                Rop[r * nt:(r + 1) * nt, s * nt:(s + 1) * nt] = dt * w[s] * (PB @ Cm)
        return -Th @ Tall @ Rop

    scale = 0.5 / np.linalg.norm(dense_A(R), 2)                 # scaled-down R: ||A||_2 = 0.5
    Rs = (R.astype(np.float64) * scale).astype(np.float32)     # the oracle takes fp32 R: A is built from the rounded R
    A = dense_A(Rs)
    assert 0.45 < np.linalg.norm(A, 2) < 0.55
    Gd = rng.standard_normal((1, n, nt)).astype(np.float32)
    b = (Tall @ Gd.astype(np.float64).reshape(-1))            # N_{-1} = T G_d
    o = oracle.marchenko(Rs, Gd, td, dt, dx, fmin, fmax, niter=K, eps=eps)
    I = np.eye(n * nt)
    closed = np.linalg.solve(I - A, (I - np.linalg.matrix_power(A, K + 1)) @ b)
    np.testing.assert_allclose(o["f2"].reshape(-1), closed, atol=1e-12 * np.abs(closed).max())
    # and each iterate is A^k b
    v = b.copy()
    for k in range(K):
        v = A @ v
        np.testing.assert_allclose(o["N_iters"][k].reshape(-1), v, atol=1e-12 * np.abs(b).max())


def test_subset_chain_fed_with_full_iterates_equals_the_full_chain_restricted():
    """Host logic of the "single step" parity harness: a proper receiver subset, fed at every step with the previous
    iterate at every source position, reproduces the full chain on that subset (iterates, accumulators, finals)."""
    n, nt, nfoc, dt, dx, eps, K = 7, 32, 2, 0.004, 10.0, 1, 5
    fmin, fmax = 20.0, 100.0
    R = (0.02 * rng.standard_normal((n, n, nt))).astype(np.float32)
    Gd = rng.standard_normal((nfoc, n, nt)).astype(np.float32)
    td = (dt * rng.uniform(5, 12, size=(nfoc, n))).astype(np.float32)
    full = oracle.marchenko(R, Gd, td, dt, dx, fmin, fmax, niter=K, eps=eps)
    recs = np.array([1, 4, 6])
    sub = oracle.SubsetChain(R[:, recs], td[:, recs], Gd[:, recs], dt, dx, fmin, fmax, eps)
    prev = T(Gd.astype(np.float64))
    for it in range(K):
        Nn = sub.step(prev)
        np.testing.assert_array_equal(Nn, full["N_iters"][it][:, recs])
        prev = full["N_iters"][it]
    for nm in ("f1plus", "f1min", "f2", "pmin"):
        np.testing.assert_array_equal(getattr(sub, nm), full[nm][:, recs])
    fin = sub.finals(full["f1plus"], full["f1min"])
    for nm in ("G", "Gplus", "Gminus"):
        np.testing.assert_array_equal(fin[nm], full[nm][:, recs])


def test_init_is_the_time_reversed_first_arrival():
    """O4 (orc_init_subset; "N_{-1} = f^+_{1,0} = G_d(-t)", 67, 74-75) on a hand-written trace: t -> -t with
    negative times stored wrapped keeps samples 0 and nt/2 in place and swaps j with nt - j; applying it twice is the
    identity; and the spectrum of the result is the conjugate of the input's (real trace), which is what a
    time reversal is, independent of any index formula."""
    g = np.array([[[1.0, 2.0, 3.0, 4.0, 5.0, 6.0, 7.0, 8.0]]], np.float32)
    np.testing.assert_array_equal(oracle.init_field(g)[0, 0], [1.0, 8.0, 7.0, 6.0, 5.0, 4.0, 3.0, 2.0])
    x = rng.standard_normal((2, 3, 64)).astype(np.float32)
    y = oracle.init_field(x)
    np.testing.assert_array_equal(oracle.init_field(y.astype(np.float32)), x.astype(np.float64))
    np.testing.assert_allclose(np.fft.fft(y), np.conj(np.fft.fft(x.astype(np.float64))), atol=1e-12)
    # the chain starts from it: f1plus = f2 = T G_d, f1min = pmin = 0, and with niter = 0 nothing else happens
    n, nt = 3, 64
    R = np.zeros((n, n, nt), np.float32)
    td = np.full((2, n), 0.1, np.float32)
    o = oracle.marchenko(R, x, td, 0.004, 10.0, 10.0, 100.0, niter=0)
    np.testing.assert_array_equal(o["f1plus"], y)
    np.testing.assert_array_equal(o["f2"], y)
    assert not o["f1min"].any() and not o["pmin"].any()
    sub = oracle.SubsetChain(R[:, [0, 2]], td[:, [0, 2]], x[:, [0, 2]], 0.004, 10.0, 10.0, 100.0)
    np.testing.assert_array_equal(sub.f1plus, y[:, [0, 2]])
    np.testing.assert_array_equal(sub.f2, y[:, [0, 2]])
    assert not sub.f1min.any() and not sub.pmin.any()


def test_general_geometry_is_the_square_scheme_on_the_union_grid():
    """orc_marchenko_geom (sources and receivers not co-located one to one; eq. (1): integral over source
    positions, evaluated at receiver positions; PAPER.md:28 keeps ns and nr apart).  Pins:
    (i) identity geometry (nshot = nrec, shot s at receiver s, trapezoid weights) IS orc_marchenko, bit for bit;
    (ii) any geometry equals the pinned SQUARE scheme on the union grid of positions, where a missing source or receiver
    is a zero row / column of R and a zero first arrival with an empty window, and the shot weights are folded into R
    (the square scheme has its own trapezoid weights) — an independent route through code that is pinned elsewhere."""
    nt, dt, dx, eps, K = 32, 0.004, 10.0, 1, 4
    fmin, fmax = 20.0, 100.0
    # (i)
    n, nfoc = 6, 2
    R = (0.02 * rng.standard_normal((n, n, nt))).astype(np.float32)
    Gd = rng.standard_normal((nfoc, n, nt)).astype(np.float32)
    td = (dt * rng.uniform(5, 12, size=(nfoc, n))).astype(np.float32)
    sq = oracle.marchenko(R, Gd, td, dt, dx, fmin, fmax, niter=K, eps=eps)
    ge = oracle.marchenko_geom(R, Gd, td, dt, oracle.weights(n, dx), np.arange(n), fmin, fmax, K, eps)
    for nm in ("N_iters", "f1plus", "f1min", "f2", "pmin", "G", "Gplus", "Gminus"):
        np.testing.assert_array_equal(ge[nm], sq[nm])
    # (ii) union grid of 9 positions; shots at S, receivers at Rc; 2 shots without a receiver, 3 receivers without a shot
    U = 9
    S = np.array([0, 1, 3, 4, 6, 8])            # positions of the 6 shots
    Rc = np.array([1, 2, 3, 5, 6, 7, 8])        # positions of the 7 receivers
    ns, nr = len(S), len(Rc)
    rec_of_shot = np.array([int(np.nonzero(Rc == p)[0][0]) if p in Rc else -1 for p in S])
    assert (rec_of_shot >= 0).sum() == 4
    Rg = (0.03 * rng.standard_normal((ns, nr, nt))).astype(np.float32)
    Gdg = rng.standard_normal((nfoc, nr, nt)).astype(np.float32)
    tdg = (dt * rng.uniform(5, 12, size=(nfoc, nr))).astype(np.float32)
    wU = oracle.weights(U, dx)
    # irregular quadrature weights of the shot grid, chosen so that folding them into R is exact in fp32: powers of two times wU
    w2 = np.array([wU[p] * 2.0 ** k for p, k in zip(S, [0, 1, -1, 0, 2, -2])])
    RU = np.zeros((U, U, nt), np.float32)
    for i, ps in enumerate(S):
        for j, pr in enumerate(Rc):
            RU[ps, pr] = Rg[i, j] * np.float32(w2[i] / wU[ps])          # exact: a power of two
    GdU = np.zeros((nfoc, U, nt), np.float32)
    tdU = np.zeros((nfoc, U), np.float32)                                 # t_d = 0: window half-width 0, trace stays zero
    GdU[:, Rc] = Gdg
    tdU[:, Rc] = tdg
    ge = oracle.marchenko_geom(Rg, Gdg, tdg, dt, w2, rec_of_shot, fmin, fmax, K, eps)
    sq = oracle.marchenko(RU, GdU, tdU, dt, dx, fmin, fmax, niter=K, eps=eps)
    scale = np.abs(sq["G"]).max()
    for nm in ("f1plus", "f1min", "f2", "pmin", "G", "Gplus", "Gminus"):
        np.testing.assert_allclose(ge[nm], sq[nm][:, Rc], atol=1e-13 * scale, rtol=0)
        off = np.setdiff1d(np.arange(U), Rc)
        if nm in ("f1plus", "f1min", "f2"):
            assert not sq[nm][:, off].any()                               # nothing lives where there is no receiver
    for k in range(K):
        np.testing.assert_allclose(ge["N_iters"][k], sq["N_iters"][k][:, Rc], atol=1e-13 * scale, rtol=0)
    assert np.abs(ge["N_iters"][-1]).max() > 1e-6 * np.abs(ge["N_iters"][0]).max() > 0


def test_image_is_the_zero_lag_of_the_convolution():
    """image[f] = dt sum_r w[r] (G^- (*) f1plus)[0]: brute force on a tiny case and numpy's FFT convolution theorem."""
    nfoc, n, nt, dt, dx = 3, 5, 16, 0.004, 10.0
    g = rng.standard_normal((nfoc, n, nt))
    p = rng.standard_normal((nfoc, n, nt))
    w = np.full(n, dx)
    w[0] = w[-1] = dx / 2
    brute = np.array([dt * sum(w[r] * sum(g[f, r, (0 - j) % nt] * p[f, r, j] for j in range(nt)) for r in range(n))
                      for f in range(nfoc)])
    lag0 = np.fft.irfft(np.fft.rfft(g) * np.fft.rfft(p), nt)[..., 0]
    got = oracle.image(g, p, dt, dx)
    np.testing.assert_allclose(got, brute, rtol=1e-13)
    np.testing.assert_allclose(got, dt * (lag0 * w).sum(axis=1), rtol=1e-12)
    # a pure delay pair: G^- = delta(t - a), f1plus = delta(t + a)  =>  image = dt * sum w
    g[:] = 0.0
    p[:] = 0.0
    g[..., 3] = 1.0
    p[..., nt - 3] = 1.0
    np.testing.assert_allclose(oracle.image(g, p, dt, dx), dt * w.sum())
