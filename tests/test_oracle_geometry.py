"""Pins for the oracle's geometry state and transform (O1, O2, O3, O6, O7).  CPU only.

What each pin holds the oracle against (never against itself):
  Jacobi            numpy.linalg.eigh (LAPACK, a different algorithm), 2x2 closed form, residuals
  subspace iter.    exact-rank-k matrix converges in one step; brute force; eigh on gapped spectra
  factor            numpy X^T X / T, trace identity, convergence to the generating covariance
  whitening         round trip (Eq. 17/19 inverts Eq. 14/18), T A_bar T = rho I and sample covariance
                    of whitened draws, explicit Kronecker products (Eq. 7-10, Eq. 15), k = d against
                    the Cholesky form of Eq. 14, dense form == low-rank form
  identity factors  codec == plain Euclidean FP8 bit for bit
  metrics           Eq. 21 against numpy
"""
import numpy as np
import pytest
import torch

import oracle
from paper_2607_07494_b200 import synth


def _rand_orth(d, rng):
    q, r = np.linalg.qr(rng.normal(size=(d, d)))
    return q * np.sign(np.diag(r))


def _spd(d, rng, lam):
    Q = _rand_orth(d, rng)
    return (Q * lam) @ Q.T, Q


# ---- Jacobi -----------------------------------------------------------------------------------------
def test_jacobi_2x2_closed_form():
    a, b, c = 2.0, 0.7, -1.0
    M, Z = oracle.jacobi_eig(np.array([[a, b], [b, c]]))
    disc = np.sqrt((a - c) ** 2 / 4 + b * b)
    assert np.allclose(M, [(a + c) / 2 + disc, (a + c) / 2 - disc], rtol=0, atol=1e-15)
    v = np.array([b, M[0] - a]); v /= np.linalg.norm(v)
    assert abs(abs(v @ Z[:, 0]) - 1) < 1e-15


@pytest.mark.parametrize("n", [1, 3, 16, 64])
def test_jacobi_against_lapack_and_residuals(n):
    rng = np.random.default_rng(n)
    lam = np.sort(rng.uniform(-1, 3, n))[::-1]
    B, _ = _spd(n, rng, lam)
    B = 0.5 * (B + B.T)
    M, Z = oracle.jacobi_eig(B)
    w = np.linalg.eigh(B)[0][::-1]
    assert np.allclose(M, w, rtol=0, atol=1e-13) and np.allclose(M, lam, atol=1e-12)
    assert np.all(np.diff(M) <= 0)
    assert np.abs(B @ Z - Z * M).max() <= 1e-13 * max(1, np.abs(B).max() * n)
    assert np.abs(Z.T @ Z - np.eye(n)).max() <= 1e-13
    assert abs(M.sum() - np.trace(B)) <= 1e-12


# ---- factor ----------------------------------------------------------------------------------------
def test_factor_accumulate_is_mean_outer_product_and_ema():
    rng = np.random.default_rng(0)
    T, d = 300, 24
    X = rng.normal(size=(T, d))
    A = oracle.factor_accumulate(X)
    assert np.allclose(A, X.T @ X / T, rtol=0, atol=1e-13)
    assert np.array_equal(A, A.T) and np.linalg.eigvalsh(A).min() > -1e-12
    assert abs(np.trace(A) - (X ** 2).sum(1).mean()) < 1e-12
    X2 = rng.normal(size=(50, d))
    A2 = oracle.factor_accumulate(X2, A, beta=0.9)
    assert np.allclose(A2, 0.9 * A + 0.1 * (X2.T @ X2 / 50), rtol=0, atol=1e-13)


def test_factor_converges_to_generating_covariance():
    d, T = 32, 20000
    X = synth.factor_samples(T, d, "cpu", 123).double().numpy()
    # the generator's covariance is Q diag(i^-2) Q^T: its spectrum must come back at O(sqrt(d/T))
    A = oracle.factor_accumulate(X)
    w = np.linalg.eigvalsh(A)[::-1]
    want = np.arange(1, d + 1.0) ** -2
    assert np.abs(w[:4] - want[:4]).max() < 5 * np.sqrt(d / T) * want[0]
    assert abs(np.trace(A) - want.sum()) < 0.05 * want.sum()


# ---- subspace iteration ------------------------------------------------------------------------------
def test_exact_rank_k_converges_in_one_step():
    rng = np.random.default_rng(4)
    d, k = 40, 5
    Q = _rand_orth(d, rng)
    lam = np.array([5.0, 3.0, 2.0, 1.0, 0.5])
    A = (Q[:, :k] * lam) @ Q[:, :k].T                            # span(A V0) = range(A) for generic V0
    b = oracle.refresh_basis(A, rng.normal(size=(d, k)), q=1, lam=1e-3)
    assert np.allclose(b.mu, lam, rtol=0, atol=1e-12)
    assert np.abs(b.U @ b.U.T - Q[:, :k] @ Q[:, :k].T).max() < 1e-12
    assert abs(b.rho - 1e-3) < 1e-15                             # zero tail + damping


def test_subspace_iteration_against_brute_force_and_lapack():
    rng = np.random.default_rng(8)
    d, k, lam_d = 48, 6, 1e-3
    spec = np.arange(1, d + 1.0) ** -2
    spec[k:] *= 0.01                                            # designed gap after k
    A, Q = _spd(d, rng, spec)
    A = 0.5 * (A + A.T)
    bf = oracle.brute_basis(A, k, lam_d)
    w, v = np.linalg.eigh(A)
    assert np.allclose(bf.mu, w[::-1][:k], rtol=0, atol=1e-14)
    Ptrue = v[:, ::-1][:, :k] @ v[:, ::-1][:, :k].T
    assert np.abs(bf.U @ bf.U.T - Ptrue).max() < 1e-12
    V0 = rng.normal(size=(d, k))
    errs = []
    for q in (1, 2, 3, 4):
        b = oracle.refresh_basis(A, V0, q, lam_d)
        assert np.abs(b.U.T @ b.U - np.eye(k)).max() < 1e-13
        errs.append(np.linalg.norm(b.U @ b.U.T - Ptrue))
    ratio = spec[k] / spec[k - 1]                               # convergence rate mu_{k+1} / mu_k
    assert errs[3] < 1e-7 and errs[1] < errs[0] * ratio * 10 and errs[2] < errs[1] * ratio * 10
    b = oracle.refresh_basis(A, V0, 6, lam_d)
    assert np.allclose(b.mu, bf.mu, rtol=1e-12) and abs(b.rho - bf.rho) < 1e-15
    assert np.allclose(np.abs(b.U), np.abs(bf.U), atol=1e-9)
    assert np.all(b.U[np.abs(b.U).argmax(0), np.arange(k)] > 0)   # sign rule
    # multipliers from their definition (S2): rho = mean tail eigenvalue + lam
    rho = (np.trace(A) - bf.mu.sum()) / (d - k) + lam_d
    assert abs(bf.rho - rho) < 1e-15
    D = np.sqrt(rho / (bf.mu + lam_d))
    assert np.allclose(bf.e, D - 1, atol=1e-15) and np.allclose(bf.ebar, 1 / D - 1, atol=1e-13)


# ---- whitening algebra -------------------------------------------------------------------------------
def _setup(m, n, kG, kA, seed, lam=1e-3):
    rng = np.random.default_rng(seed)
    A, _ = _spd(n, rng, np.arange(1, n + 1.0) ** -2)
    G, _ = _spd(m, rng, np.arange(1, m + 1.0) ** -2)
    A, G = 0.5 * (A + A.T), 0.5 * (G + G.T)
    bA = oracle.brute_basis(A, kA, lam)
    bG = oracle.brute_basis(G, kG, lam)
    W = rng.normal(size=(m, n))
    return rng, A, G, bA, bG, W


def _abar(b, lam):
    d, k = b.U.shape
    return (b.U * (b.mu + lam)) @ b.U.T + b.rho * (np.eye(d) - b.U @ b.U.T)


def test_roundtrip_without_quantisation_reproduces_W():
    rng, A, G, bA, bG, W = _setup(20, 28, 4, 6, 1)
    for UG, UA in [(bG, bA), (None, bA), (bG, None), (None, None)]:
        wt = oracle.whiten_lowrank(W, UG.U if UG else None, UG.e if UG else None,
                                   UA.U if UA else None, UA.e if UA else None)
        back = oracle.whiten_lowrank(wt, UG.U if UG else None, UG.ebar if UG else None,
                                     UA.U if UA else None, UA.ebar if UA else None)
        assert np.abs(back - W).max() < 1e-12
        if UG is None and UA is None:
            assert np.array_equal(wt, W)


def test_dense_form_equals_lowrank_form_and_T_inverse():
    rng, A, G, bA, bG, W = _setup(20, 28, 4, 6, 2)
    TA, TG = oracle.build_T(bA.U, bA.e), oracle.build_T(bG.U, bG.e)
    assert np.allclose(TA, np.eye(28) + (bA.U * bA.e) @ bA.U.T, atol=1e-15)
    assert np.abs(TA @ oracle.build_T(bA.U, bA.ebar) - np.eye(28)).max() < 1e-13
    lr = oracle.whiten_lowrank(W, bG.U, bG.e, bA.U, bA.e)
    assert np.abs(oracle.whiten_dense(W, TG, TA) - lr).max() < 1e-13
    assert np.abs(TG @ W @ TA - lr).max() < 1e-13                     # numpy matmul, independent
    assert np.abs(oracle.whiten_dense(W, None, TA) - oracle.whiten_lowrank(W, None, None, bA.U, bA.e)).max() < 1e-13
    assert np.abs(W @ TA - oracle.whiten_lowrank(W, None, None, bA.U, bA.e)).max() < 1e-13
    assert np.abs(TG @ W - oracle.whiten_lowrank(W, bG.U, bG.e, None, None)).max() < 1e-13


def test_T_whitens_the_damped_lowrank_model():
    lam = 1e-3
    rng, A, G, bA, bG, W = _setup(12, 40, 3, 8, 3, lam)
    TA = oracle.build_T(bA.U, bA.e)
    Abar = _abar(bA, lam)
    assert np.abs(TA @ Abar @ TA - bA.rho * np.eye(40)).max() < 1e-15 + 1e-12 * bA.rho   # exactly rho I
    # rows drawn from N(0, A_bar) come out with sample covariance ~ rho I (ellipsoid -> ball, Eq. 11-13)
    N = 40000
    L = np.linalg.cholesky(Abar)
    rows = rng.normal(size=(N, 40)) @ L.T
    wt = oracle.whiten_lowrank(rows, None, None, bA.U, bA.e)
    C = wt.T @ wt / N / bA.rho
    assert np.abs(C - np.eye(40)).max() < 6 / np.sqrt(N) * 2
    C0 = rows.T @ rows / N / bA.rho                                  # before: strongly anisotropic
    assert np.linalg.cond(C0) > 50 and np.linalg.cond(C) < 1.3


def test_kronecker_identities_eq7_to_eq15():
    lam = 1e-2
    rng, A, G, bA, bG, W = _setup(5, 7, 2, 3, 4, lam)
    TA, TG = oracle.build_T(bA.U, bA.e), oracle.build_T(bG.U, bG.e)
    vec = lambda X: X.reshape(-1, order="F")                          # column-major vec
    wt = oracle.whiten_lowrank(W, bG.U, bG.e, bA.U, bA.e)
    assert np.abs(vec(wt) - np.kron(TA, TG) @ vec(W)).max() < 1e-13   # Eq. 15, T symmetric
    # Eq. 7-10 with the symmetric roots S = A_bar^(1/2) = sqrt(rho) T^-1:
    #   vec(dW)^T (A_bar kron G_bar) vec(dW) = tr(A_bar dW^T G_bar dW) = ||S_G dW S_A||_F^2
    Abar, Gbar = _abar(bA, lam), _abar(bG, lam)
    dW = rng.normal(size=(5, 7))
    lhs = vec(dW) @ np.kron(Abar, Gbar) @ vec(dW)
    mid = np.trace(Abar @ dW.T @ Gbar @ dW)
    un = oracle.whiten_lowrank(dW, bG.U, bG.ebar, bA.U, bA.ebar)      # T_G^-1 dW T_A^-1
    rhs = bA.rho * bG.rho * (un ** 2).sum()
    assert abs(lhs - mid) < 1e-12 * abs(lhs) and abs(lhs - rhs) < 1e-12 * abs(lhs)


def test_full_rank_matches_cholesky_form_of_eq14():
    lam = 1e-3
    rng, A, G, _, _, W = _setup(9, 11, 1, 1, 5, lam)
    bA, bG = oracle.brute_basis(A, 11, lam), oracle.brute_basis(G, 9, lam)
    assert abs(bA.rho - (bA.mu[-1] + lam)) < 1e-18
    wt = oracle.whiten_lowrank(W, bG.U, bG.e, bA.U, bA.e) / np.sqrt(bA.rho * bG.rho)
    LA, LG = np.linalg.cholesky(A + lam * np.eye(11)), np.linalg.cholesky(G + lam * np.eye(9))
    ref = np.linalg.solve(LG, W) @ np.linalg.inv(LA).T               # L_G^-1 W L_A^-T  (Eq. 14)
    s1, s2 = np.linalg.svd(wt, compute_uv=False), np.linalg.svd(ref, compute_uv=False)
    assert np.allclose(s1, s2, rtol=1e-9)                            # equal up to orthogonal factors
    # and T_A itself is sqrt(rho) (A + lam I)^(-1/2)
    w, v = np.linalg.eigh(A + lam * np.eye(11))
    assert np.abs(oracle.build_T(bA.U, bA.e) - np.sqrt(bA.rho) * (v / np.sqrt(w)) @ v.T).max() < 1e-10


def test_isotropic_factors_reduce_to_euclidean_fp8():
    rng = np.random.default_rng(6)
    m, n, k = 24, 40, 5
    W = rng.normal(size=(m, n)).astype(np.float32)
    bA = oracle.refresh_basis(2.5 * np.eye(n), rng.normal(size=(n, k)), 2, 1e-3)
    bG = oracle.refresh_basis(0.3 * np.eye(m), rng.normal(size=(m, k)), 2, 1e-3)
    assert np.abs(bA.e).max() < 1e-14 and np.abs(bG.ebar).max() < 1e-14
    for fmt in (oracle.E4M3, oracle.E5M2):
        c1, s1, x1 = oracle.encode(W.astype(np.float64), bG, bA, fmt)
        c0, s0, x0 = oracle.encode(W.astype(np.float64), None, None, fmt)
        assert np.array_equal(x1, W) and np.array_equal(c1, c0) and np.array_equal(s1, s0)


def test_metrics_eq21():
    rng = np.random.default_rng(7)
    g, h = rng.normal(size=500), rng.normal(size=500)
    mt = oracle.metrics(h, g)
    assert np.isclose(mt["RelL2"], np.linalg.norm(h - g) / np.linalg.norm(g), rtol=1e-14)
    assert np.isclose(mt["Cos"], h @ g / np.linalg.norm(h) / np.linalg.norm(g), rtol=1e-13)
    assert mt["MaxErr"] == np.abs(h - g).max() and np.isclose(mt["MSE"], ((h - g) ** 2).mean(), rtol=1e-14)


# ---- config 0 end to end on the oracle alone ---------------------------------------------------------
def test_config0_pipeline_properties():
    cfg = synth.config(0)
    t = cfg.tensors[0]
    G = synth.tensor_gradient(cfg, t, "cpu")
    X = synth.tensor_factor_samples(cfg, t, "in", "cpu").double().numpy()
    Dl = synth.tensor_factor_samples(cfg, t, "out", "cpu").double().numpy()
    A, Gf = oracle.factor_accumulate(X), oracle.factor_accumulate(Dl)
    bA = oracle.refresh_basis(A, synth.tensor_start_basis(cfg, t, "in", "cpu").double().numpy(), 8, cfg.damping)
    bG = oracle.refresh_basis(Gf, synth.tensor_start_basis(cfg, t, "out", "cpu").double().numpy(), 8, cfg.damping)
    # Ritz values never exceed the true eigenvalues (Cauchy interlacing) and approach them from below
    wa = np.linalg.eigvalsh(A)[::-1][: t.rank]
    assert np.all(bA.mu <= wa * (1 + 1e-12)) and np.all(bA.mu[:8] >= wa[:8] * 0.99)
    payloads = []
    for r in range(cfg.R):
        Gr = synth.tensor_rank_gradient(cfg, t, G, r).double().numpy()
        c, s, _ = oracle.encode(Gr, bG, bA)
        payloads.append((c, s))
    out = oracle.reduce_decoded([p[0] for p in payloads], [p[1] for p in payloads], bG, bA)
    mean = sum(synth.tensor_rank_gradient(cfg, t, G, r).double().numpy() for r in range(cfg.R)) / cfg.R
    mt = oracle.metrics(out, mean)
    # An FP8 round trip, not garbage.  The config draws G independently of the factors (DESIGN.md
    # reading S15), so unwhitening amplifies the isotropic FP8 noise along the top-k directions by
    # (mu_i + lam) / rho: ~0.019 per-side-whitened error * ~6 here.  No fidelity gain is expected.
    assert mt["RelL2"] < 0.2 and mt["Cos"] > 0.99


# ---- sampled-output routines (full-size parity helpers) pinned against the whole-matrix forms and closed forms ------
def test_sampled_outputs_agree_with_whole_matrix_forms_and_closed_forms():
    rng = np.random.default_rng(11)
    m, n, kG, kA = 40, 56, 5, 7
    W = rng.normal(size=(m, n))
    UG = np.linalg.qr(rng.normal(size=(m, kG)))[0]
    UA = np.linalg.qr(rng.normal(size=(n, kA)))[0]
    eG, eA = rng.uniform(-0.9, 3.0, kG), rng.uniform(-0.9, 3.0, kA)
    ii, jj = rng.integers(0, m, 64), rng.integers(0, n, 64)
    # (a) against the low-rank whole-matrix form (two independent oracle forms of Eq. 14 must agree), all side combinations
    for ug, ua in ((UG, UA), (UG, None), (None, UA), (None, None)):
        full = oracle.whiten_lowrank(W, ug, eG if ug is not None else None, ua, eA if ua is not None else None)
        got = oracle.whiten_samples(W, ii, jj, ug, eG if ug is not None else None, ua, eA if ua is not None else None)
        assert np.abs(got - full[ii, jj]).max() <= 1e-12 * np.abs(full).max()
    # (b) against the explicit dense T matrices built with numpy (Eq. 14)
    TG = np.eye(m) + UG @ np.diag(eG) @ UG.T
    TA = np.eye(n) + UA @ np.diag(eA) @ UA.T
    assert np.abs(oracle.whiten_samples(W, ii, jj, UG, eG, UA, eA) - (TG @ W @ TA)[ii, jj]).max() <= 1e-12 * np.abs(W).max() * 20
    # (c) a transposed-operand mistake shows: a matrix with one non-zero element and rank-one factors has a closed form
    W1 = np.zeros((m, n)); W1[3, 9] = 2.0
    want = 2.0 * TG[ii, 3] * TA[9, jj]
    assert np.abs(oracle.whiten_samples(W1, ii, jj, UG, eG, UA, eA) - want).max() <= 1e-13
    # factor entries: the whole-matrix routine, and a closed form (one-hot samples: A = diag(counts) / T)
    X = rng.normal(size=(33, 12))
    fi, fj = rng.integers(0, 12, 40), rng.integers(0, 12, 40)
    assert np.abs(oracle.factor_entries(X, fi, fj) - oracle.factor_accumulate(X)[fi, fj]).max() <= 1e-14
    onehot = np.eye(12)[[0, 0, 5, 7, 7, 7]]
    assert np.allclose(oracle.factor_entries(onehot, [0, 5, 7, 0], [0, 5, 7, 5]), [2 / 6, 1 / 6, 3 / 6, 0.0], atol=1e-15)
