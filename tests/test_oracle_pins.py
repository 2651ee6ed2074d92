"""Pins for the CPU oracle (oracle/gsr_oracle.c) against things other than itself:
a hand-worked fixture, dense numpy linear algebra, closed forms, invariants the paper states,
and scipy's independent LSQR (same published algorithm).  CPU only."""
import dataclasses
import os

import numpy as np
import pytest
import scipy.sparse as sp
import scipy.sparse.linalg as spla

import oracle
from paper_2308_00778_b200 import synth
from helpers import dense, make_b, np_inputs, oracle_system

GOLD = os.path.join(os.path.dirname(__file__), "golden")


# ----------------------------------------------------------------------------- fixture
def _parse_hand():
    rows, kv = [], {}
    for line in open(os.path.join(GOLD, "hand_system.txt")):
        line = line.split("#")[0].strip()
        if not line:
            continue
        tok = line.split()
        if tok[0] == "row":
            a, b_, c = line[3:].split("|")
            ia, iatt = map(int, a.split())
            rows.append((ia, iatt, list(map(int, b_.split())), c.strip()))
        else:
            kv[tok[0]] = [float(t) for t in tok[1:]]
    return rows, kv


def test_hand_worked_fixture():
    """PAPER.md:78-80 + Alg. 2 index expressions, worked by hand (tests/golden/hand_system.txt)."""
    rows, kv = _parse_hand()
    rule = {"ones": lambda k: 1.0, "kplus1": lambda k: k + 1.0, "altsign": lambda k: (-1.0) ** k}
    V = np.array([[rule[r[3]](k) for k in range(24)] for r in rows])
    S = oracle.OracleSystem(int(kv["n_stars"][0]), int(kv["n_dof_att"][0]), int(kv["n_instr"][0]), V,
                            [r[0] for r in rows], [r[1] for r in rows], [r[2] for r in rows])
    assert S.n == 32
    assert [S.col(1, k) for k in range(24)] == [int(c) for c in kv["cols1"]]
    x = np.arange(1, 33, dtype=np.float64)
    y, ab = S.aprod1(x, np.array(kv["aprod1_yin"]), want_abs=True)
    assert y.tolist() == kv["aprod1_yout"]
    # all terms of rows 0 and 1 are positive: the abs bound is |y_in| + the sum itself
    assert ab[0] == 1000 + 428 and ab[1] == 2000 + 7039
    xo = S.aprod2(np.array(kv["aprod2_y"]), np.zeros(32))
    assert xo.tolist() == kv["aprod2_xout"]


# ----------------------------------------------------------------------------- structure + dense
@pytest.mark.parametrize("seed", [0, 1])
@pytest.mark.parametrize("ncon", [0, 3])
def test_dense_expansion_and_structure(seed, ncon):
    cfg = synth.mini(seed=seed, n_con=ncon, con_nnz=7 if ncon else 0)
    S, d = oracle_system(cfg)
    A = dense(S)
    m, ns, nd, ni = S.m, cfg.n_stars, cfg.n_dof_att, cfg.n_instr
    off_att, off_instr, off_glob = 5 * ns, 5 * ns + 3 * nd, 5 * ns + 3 * nd + ni
    assert S.n == off_glob + 1 == cfg.n
    # at most N_par = 24 stored coefficients per row; here exactly 24 distinct columns
    assert ((A[:m] != 0).sum(axis=1) == 24).all()
    star = d["matrixIndexAstro"] // 5
    for i in range(m):
        nz = np.nonzero(A[i])[0]
        # block-diagonal astrometric part, N_Astro=5 columns per star block
        assert nz[:5].tolist() == list(range(5 * star[i], 5 * star[i] + 5))
        # N_Att=12 as 3 blocks of 4 consecutive elements, blocks N_DFA apart
        att = nz[5:17].reshape(3, 4)
        assert (np.diff(att, axis=1) == 1).all()
        assert (np.diff(att[:, 0]) == nd).all()
        assert off_att <= att[0, 0] and att[0, 3] < off_att + nd
        # instrumental: 6 columns "without a particular scheme" inside the instrumental range
        assert ((nz[17:23] >= off_instr) & (nz[17:23] < off_glob)).all()
        assert sorted(nz[17:23] - off_instr) == sorted(d["instrCol"][i].tolist())
        # one global column (gamma), the last unknown
        assert nz[23] == off_glob
    # the astro part of A is block diagonal: rows of star s only touch block s
    blocks = A[:m, :off_att].reshape(m, ns, 5)
    assert (np.abs(blocks).sum(axis=2) != 0).sum(axis=1).max() == 1
    # aprod1 / aprod2 against numpy's dense products
    rng = np.random.default_rng(seed)
    x, y0 = rng.standard_normal(S.n), rng.standard_normal(S.m_tot)
    y, ab = S.aprod1(x, y0, want_abs=True)
    ref_ab = np.abs(y0) + np.abs(A) @ np.abs(x)
    np.testing.assert_allclose(ab, ref_ab, rtol=1e-13)
    assert (np.abs(y - (y0 + A @ x)) <= 1e-14 * ref_ab).all()
    yv, x0 = rng.standard_normal(S.m_tot), rng.standard_normal(S.n)
    xo, ab2 = S.aprod2(yv, x0, want_abs=True)
    ref_ab2 = np.abs(x0) + np.abs(A).T @ np.abs(yv)
    np.testing.assert_allclose(ab2, ref_ab2, rtol=1e-13)
    assert (np.abs(xo - (x0 + A.T @ yv)) <= 1e-14 * ref_ab2).all()
    # accumulate semantics (Eq. 2-3 "+="): zero input vector leaves the target untouched
    assert (S.aprod1(np.zeros(S.n), y0) == y0).all()
    assert (S.aprod2(np.zeros(S.m_tot), x0) == x0).all()


def test_adjoint_identity_tiny_config():
    """<A x, y> = <x, A^T y> on BASELINE configs[0] (100,000 rows)."""
    cfg = synth.tiny()
    S, d = oracle_system(cfg)
    rng = np.random.default_rng(5)
    x, y = rng.standard_normal(S.n), rng.standard_normal(S.m_tot)
    Ax = S.aprod1(x, np.zeros(S.m_tot))
    Aty = S.aprod2(y, np.zeros(S.n))
    lhs, rhs = Ax @ y, x @ Aty
    assert abs(lhs - rhs) <= 1e-13 * np.linalg.norm(Ax) * np.linalg.norm(y)


def test_skewed_generator_shape():
    cfg = dataclasses.replace(synth.skewed(), n_stars=300, n_dof_att=5000, n_instr=500)
    S, d = oracle_system(cfg)
    cnt = np.diff(d["rowptr"])
    assert cnt.min() >= 10 and cnt.max() <= 2000 and S.m == cnt.sum()
    assert (np.diff(d["matrixIndexAstro"]) >= 0).all()
    st = d["matrixIndexAstro"] // 5
    same = st[1:] == st[:-1]
    assert (np.diff(d["matrixIndexAtt"])[same] >= 0).all()      # time-sorted within a star
    ic = np.sort(d["instrCol"], axis=1)
    assert (ic[:, 1:] != ic[:, :-1]).all()


# ----------------------------------------------------------------------------- Eq. 4
def test_norm_eq4():
    rng = np.random.default_rng(0)
    a = rng.standard_normal(1000)
    assert abs(oracle.norm(a) - np.linalg.norm(a)) <= 4e-16 * np.linalg.norm(a) * 8
    assert oracle.norm(np.zeros(7)) == 0.0
    assert oracle.norm(np.array([-3.0, 4.0])) == 5.0
    # the point of the max-scaled form ("not to loose in numerical precision"):
    assert oracle.norm(np.array([3e200, -4e200])) == pytest.approx(5e200, rel=1e-15)
    assert oracle.norm(np.array([3e-200, 4e-200])) == pytest.approx(5e-200, rel=1e-15)


# ----------------------------------------------------------------------------- preconditioning
def test_precondition_unit_columns():
    cfg = synth.mini(seed=3, n_stars=6, obs=9, n_dof_att=12, n_instr=400, n_con=2, con_nnz=5)
    S, d = oracle_system(cfg)
    A0 = dense(S)
    p = S.precondition()
    A1 = dense(S)
    nrm0 = np.linalg.norm(A0, axis=0)
    empty = nrm0 == 0
    assert empty.any(), "fixture should contain unused instrumental columns"
    assert (p[empty] == 1.0).all()
    np.testing.assert_allclose(p[~empty], 1.0 / nrm0[~empty], rtol=1e-14)
    np.testing.assert_allclose(np.linalg.norm(A1, axis=0)[~empty], 1.0, rtol=0, atol=8 * 2.3e-16)
    assert abs((A1 ** 2).sum() - (~empty).sum()) < 1e-12 * (~empty).sum()
    np.testing.assert_allclose(A1, A0 * p[None, :], rtol=1e-15)


# ----------------------------------------------------------------------------- LSQR
def _csr(S):
    return sp.csr_matrix(dense(S))


@pytest.mark.parametrize("precond", [False, True])
@pytest.mark.parametrize("ncon", [0, 4])
def test_lsqr_matches_dense_least_squares(precond, ncon):
    cfg = synth.mini(seed=11, n_con=ncon, con_nnz=9 if ncon else 0)
    S, d = oracle_system(cfg)
    A0 = dense(S)
    b = make_b(S, d)
    if precond:
        S.precondition()
    r = S.lsqr(b, 10 * S.n, 1e-15, 1e-15)
    x_ref = np.linalg.lstsq(A0, b, rcond=None)[0]
    cond = np.linalg.cond(A0 * (S.p[None, :] if precond else 1.0))
    assert r.istop in (1, 2, 4, 5)
    assert np.linalg.norm(r.x - x_ref) <= 1e-10 * cond * np.linalg.norm(x_ref)
    # planted solution is recovered up to the noise level (sigma = 1e-3)
    assert np.linalg.norm(r.x - d["x_true"]) <= 0.05 * np.linalg.norm(d["x_true"])


def test_covariances_against_krylov_closed_form():
    """Covariances of couples of unknowns (Alg. 1 l.26-27; R26): the off-diagonal entries of
    sum_{i<=k} d_i d_i^T = V_k (B_k^T B_k)^-1 V_k^T (dense, re-orthogonalised Golub-Kahan; nothing of the LSQR
    recurrences; at k = n that matrix is (A'^T A')^-1, checked on the dense side), scaled by the TRUE residual of the
    dense Krylov solution over (m - n) and by p_i p_j, while the oracle's Lanczos vectors are still orthogonal
    (k <= 20, as for the variances).  Also: cov(i, i) = se_i^2, cov(i, j) = cov(j, i), |cov(i, j)| <= se_i se_j
    (the estimate is positive semi-definite), and a solve with couples returns x / se bit for bit as one without."""
    cfg = synth.mini(seed=9, n_stars=3, obs=16, n_dof_att=5, n_instr=6)
    S, d = oracle_system(cfg)
    b = make_b(S, d)
    p = S.precondition()
    A = dense(S)
    n = S.n
    B, V, beta = _golub_kahan_reorth(A, b, n)
    np.testing.assert_allclose(V @ np.linalg.inv(B.T @ B) @ V.T, np.linalg.inv(A.T @ A), rtol=0, atol=1e-9)
    rng = np.random.default_rng(5)
    pi = np.concatenate([rng.integers(0, n, 40), np.arange(6)])
    pj = np.concatenate([rng.integers(0, n, 40), np.arange(6)])        # the last six couples are (i, i)
    for k in (1, 2, 5, 10, 20):
        Bk, Vk = B[:k + 1, :k], V[:, :k]
        e1 = np.zeros(k + 1)
        e1[0] = beta
        zk = Vk @ np.linalg.lstsq(Bk, e1, rcond=None)[0]
        C_ref = Vk @ np.linalg.inv(Bk.T @ Bk) @ Vk.T
        s2 = np.linalg.norm(b - A @ zk) ** 2 / (S.m_tot - n)
        cov_ref = p[pi] * p[pj] * s2 * C_ref[pi, pj]
        rk = S.lsqr(b, k, 0.0, 0.0, pairs=(pi, pj))
        scale = p[pi] * p[pj] * s2 * np.sqrt(C_ref[pi, pi] * C_ref[pj, pj])      # |cov| <= this (Cauchy-Schwarz)
        assert np.all(np.abs(rk.cov - cov_ref) <= 1e-9 * scale), (k, np.max(np.abs(rk.cov - cov_ref) / scale))
        np.testing.assert_allclose(rk.cov[-6:], rk.se[:6] ** 2, rtol=1e-13)
        assert np.all(np.abs(rk.cov) <= rk.se[pi] * rk.se[pj] * (1 + 1e-12))
        r0 = S.lsqr(b, k, 0.0, 0.0)
        assert np.array_equal(r0.x, rk.x) and np.array_equal(r0.se, rk.se) and r0.itn == rk.itn
        rt = S.lsqr(b, k, 0.0, 0.0, pairs=(pj, pi))
        assert np.array_equal(rt.cov, rk.cov)
    assert (cov_ref[:40] < 0).any() and (cov_ref[:40] > 0).any()    # real off-diagonal entries of both signs were compared


def test_lsqr_planted_noiseless():
    cfg = dataclasses.replace(synth.mini(seed=2), noise_sigma=0.0)
    S, d = oracle_system(cfg)
    b = make_b(S, d)
    S.precondition()
    r = S.lsqr(b, 2000, 1e-14, 1e-14)
    assert r.istop in (1, 4)
    assert np.linalg.norm(r.x - d["x_true"]) <= 1e-10 * np.linalg.norm(d["x_true"])


@pytest.mark.parametrize("tol,conlim,itnlim", [(1e-14, 0.0, 5000), (1e-8, 1e8, 5000), (0.0, 0.0, 25),
                                               (0.0, 0.0, 5000)])
def test_lsqr_matches_scipy(tol, conlim, itnlim):
    """scipy.sparse.linalg.lsqr is an independent implementation of the same published
    algorithm with the same istop codes.  The four cases end with istop 2, 2, 7 and 5: with
    atol = btol = 0 and no iteration limit in reach only the rounding-floor tests are left, and
    1 + test2 <= 1 (istop 5) fires first -- the one branch no constructed case reaches."""
    cfg = synth.mini(seed=4, n_stars=30, obs=14, n_dof_att=16, n_instr=12, n_con=3, con_nnz=6)
    S, d = oracle_system(cfg)
    b = make_b(S, d)
    S.precondition()
    A = _csr(S)
    r = S.lsqr(b, itnlim, tol, tol, conlim)
    z, istop, itn, r1norm, _, anorm, acond, arnorm, xnorm, var = spla.lsqr(
        A, b, atol=tol, btol=tol, conlim=conlim, iter_lim=itnlim, calc_var=True)
    assert r.istop == istop
    assert r.istop == {(1e-14, 5000): 2, (1e-8, 5000): 2, (0.0, 25): 7, (0.0, 5000): 5}[(tol, itnlim)]
    assert abs(r.itn - itn) <= 1
    if r.itn == itn:
        assert np.linalg.norm(r.x - S.p * z) <= 1e-12 * np.linalg.norm(z)
        for mine, theirs in ((r.rnorm, r1norm), (r.xnorm, xnorm)):
            assert mine == pytest.approx(theirs, rel=1e-9)
        # alpha_k, beta_k of late iterations (after the Krylov space is numerically exhausted)
        # amplify rounding differences between two implementations, and anorm / acond sum
        # them: bit-level agreement only away from the rounding floor (R19).
        # The istop-5 case runs ~50 iterations beyond the floor: there the two agree to percent level only.
        loose = 1e-9 if itnlim == 25 else (1e-5 if tol > 0.0 else 2e-2)
        for mine, theirs in ((r.anorm, anorm), (r.acond, acond)):
            assert mine == pytest.approx(theirs, rel=loose)
        assert r.arnorm == pytest.approx(arnorm, rel=1e-6, abs=1e-12 * anorm * r1norm)
        if itnlim == 25:     # away from the rounding floor var is reproducible
            se_ref = S.p * np.sqrt(var) * r1norm / np.sqrt(S.m_tot - S.n)
            np.testing.assert_allclose(r.se, se_ref, rtol=1e-9)


def test_lsqr_scalar_estimates_track_true_quantities():
    cfg = synth.mini(seed=8)
    S, d = oracle_system(cfg)
    b = make_b(S, d)
    S.precondition()
    A = dense(S)
    nnzcols = (np.abs(A).sum(axis=0) > 0).sum()
    full = S.lsqr(b, 40, 0.0, 0.0, want_trace=True)
    assert full.istop == 7 and full.itn == 40
    tr = full.trace
    assert (np.diff(tr[:, 0]) <= 1e-14 * tr[0, 0]).all()          # rnorm non-increasing
    assert (np.diff(tr[:, 2]) >= 0).all()                          # anorm non-decreasing
    assert tr[-1, 2] <= np.sqrt(nnzcols) * (1 + 1e-12)             # anorm <= ||A'||_F
    for k in (1, 2, 5, 17, 40):
        rk = S.lsqr(b, k, 0.0, 0.0)
        z = rk.x / S.p
        res = b - A @ z
        assert rk.rnorm == pytest.approx(np.linalg.norm(res), rel=1e-10)
        assert abs(rk.arnorm - np.linalg.norm(A.T @ res)) <= 1e-10 * rk.anorm * rk.rnorm
        assert rk.xnorm == pytest.approx(np.linalg.norm(z), rel=1e-10)
        np.testing.assert_allclose([rk.rnorm, rk.arnorm, rk.anorm, rk.acond, rk.xnorm], tr[k - 1], rtol=0, atol=0)


def test_lsqr_istop_codes():
    cfg = synth.mini(seed=6)
    S, d = oracle_system(cfg)
    b_noisy = make_b(S, d)
    S.precondition()
    # b = 0 -> istop 0, x = 0, itn = 0
    r = S.lsqr(np.zeros(S.m_tot), 10, 1e-8, 1e-8)
    assert (r.istop, r.itn) == (0, 0) and not r.x.any()
    # itnlim -> 7
    assert S.lsqr(b_noisy, 3, 0.0, 0.0).istop == 7
    # noisy over-determined -> least-squares stop 2
    assert S.lsqr(b_noisy, 5000, 1e-10, 1e-10).istop == 2
    # consistent system -> 1
    cfg0 = dataclasses.replace(cfg, noise_sigma=0.0)
    S0, d0 = oracle_system(cfg0)
    b0 = make_b(S0, d0)
    S0.precondition()
    assert S0.lsqr(b0, 5000, 1e-10, 1e-10).istop == 1
    # conlim -> 3: two nearly parallel instrumental columns make cond(A') huge
    V = d["values"].copy()
    ic = d["instrCol"].copy()
    ic[:, 0], ic[:, 1] = 0, 1
    V[:, 18] = V[:, 17] * (1 + 1e-9 * np.arange(V.shape[0]) / V.shape[0])
    S3 = oracle.OracleSystem(cfg.n_stars, cfg.n_dof_att, cfg.n_instr, V, d["matrixIndexAstro"],
                             d["matrixIndexAtt"], ic)
    S3.precondition()
    assert S3.lsqr(b_noisy, 5000, 1e-13, 1e-13, conlim=10.0).istop == 3


def _golub_kahan_reorth(A, b, k):
    """Textbook Golub-Kahan lower bidiagonalisation A V_k = U_{k+1} B_k with full (twice-applied)
    re-orthogonalisation -- written from the definition, dense numpy, no LSQR recurrences."""
    m, n = A.shape
    U, V, B = np.zeros((m, k + 1)), np.zeros((n, k)), np.zeros((k + 1, k))
    beta = np.linalg.norm(b)
    U[:, 0] = b / beta
    for j in range(k):
        v = A.T @ U[:, j] - (B[j, j - 1] * V[:, j - 1] if j else 0.0)
        for _ in range(2):
            v -= V[:, :j] @ (V[:, :j].T @ v)
        B[j, j] = np.linalg.norm(v)
        V[:, j] = v / B[j, j]
        u = A @ V[:, j] - B[j, j] * U[:, j]
        for _ in range(2):
            u -= U[:, :j + 1] @ (U[:, :j + 1].T @ u)
        B[j + 1, j] = np.linalg.norm(u)
        U[:, j + 1] = u / B[j + 1, j]
    return B, V, beta


def test_x_and_se_against_krylov_closed_form():
    """Paige & Saunders: x_k = V_k argmin|B_k y - beta e1| and sum_{i<=k} d_i d_i^T =
    V_k (B_k^T B_k)^-1 V_k^T, so var_k is the diagonal of that matrix; at k = n it is
    diag((A'^T A')^-1).  The oracle's recurrences (no re-orthogonalisation) must agree with
    the closed form while the Lanczos vectors are still orthogonal (k <= 20 here), and can
    never exceed diag((A'^T A')^-1) (Loewner order of a compression)."""
    cfg = synth.mini(seed=9, n_stars=3, obs=16, n_dof_att=5, n_instr=6)
    S, d = oracle_system(cfg)
    b = make_b(S, d)
    p = S.precondition()
    A = dense(S)
    assert np.linalg.matrix_rank(A) == S.n
    full = np.diag(np.linalg.inv(A.T @ A))
    B, V, beta = _golub_kahan_reorth(A, b, S.n)
    np.testing.assert_allclose(np.diag(V @ np.linalg.inv(B.T @ B) @ V.T), full, rtol=1e-10)
    prev = np.zeros(S.n)
    for k in (1, 2, 5, 10, 20):
        Bk, Vk = B[:k + 1, :k], V[:, :k]
        e1 = np.zeros(k + 1)
        e1[0] = beta
        zk = Vk @ np.linalg.lstsq(Bk, e1, rcond=None)[0]
        var_ref = np.diag(Vk @ np.linalg.inv(Bk.T @ Bk) @ Vk.T)
        rk = S.lsqr(b, k, 0.0, 0.0)
        assert (rk.istop, rk.itn) == (7, k)
        var = (rk.se / p / rk.rnorm * np.sqrt(S.m_tot - S.n)) ** 2
        assert np.linalg.norm(rk.x / p - zk) <= 1e-12 * np.linalg.norm(zk)
        np.testing.assert_allclose(var, var_ref, rtol=1e-9)
        # the scale of se, with nothing taken from the oracle: the TRUE residual of the dense Krylov solution
        # over sqrt(m - n) (m_tot > n here), times p (Alg. 1 l.27)
        se_ref = p * np.sqrt(var_ref) * np.linalg.norm(b - A @ zk) / np.sqrt(S.m_tot - S.n)
        np.testing.assert_allclose(rk.se, se_ref, rtol=1e-9)
        assert (var <= full * (1 + 1e-9)).all()
        assert (var >= prev * (1 - 1e-12)).all()     # non-decreasing in the iteration count
        prev = var


# ----------------------------------------------------------------------------- last corners
def _dense24(A, con=None):
    """Any dense m x 24 matrix IS a Gaia-shaped system: one star (5 astro columns), N_DFA = 4 (3 x 4 attitude
    columns, start 0), 6 instrument columns 0..5, gamma: every row touches all 24 columns exactly once."""
    m = A.shape[0]
    return oracle.OracleSystem(1, 4, 6, A, np.zeros(m, np.int64), np.zeros(m, np.int64),
                               np.tile(np.arange(6, dtype=np.int32), (m, 1)))


def test_dense24_column_map_is_identity():
    A = np.arange(3 * 24, dtype=np.float64).reshape(3, 24) + 1
    S = _dense24(A)
    assert S.n == 24 and [S.col(1, k) for k in range(24)] == list(range(24))
    x = np.linspace(-1, 1, 24)
    np.testing.assert_allclose(S.aprod1(x, np.zeros(3)), A @ x, rtol=1e-14)


def test_istop4_consistent_system_solved_to_machine_precision():
    """atol = btol = 0 on a consistent system: the residual reaches the rounding floor and the only test that can
    fire is 1 + test1/(1 + anorm*xnorm/bnorm) <= 1, i.e. istop 4 (test1 <= rtol = 0 needs rnorm == 0 exactly).
    Pin: scipy's LSQR (same published algorithm) stops with 4 within one iteration of the oracle, and the
    solution is the planted one."""
    rng = np.random.default_rng(2)
    A = rng.standard_normal((40, 24))
    xt = rng.standard_normal(24)
    b = A @ xt
    r = _dense24(A).lsqr(b, 500, 0.0, 0.0)
    rs = spla.lsqr(A, b, atol=0.0, btol=0.0, conlim=0.0, iter_lim=500)
    assert r.istop == 4 == rs[1]
    assert abs(r.itn - rs[2]) <= 1
    assert np.linalg.norm(r.x - xt) <= 1e-12 * np.linalg.norm(xt)
    assert r.rnorm <= 1e-13 * np.linalg.norm(b)


def test_istop6_condition_estimate_exceeds_one_over_eps():
    """A 19 x 24 matrix of rank 11 with 4 singular values in [0.5, 1] and 7 near 10^-15.66: the Krylov process
    resolves the small cluster while A^T r is still far from zero, so acond = anorm*sqrt(ddnorm) passes 1/eps
    (1 + 1/acond <= 1, istop 6) before test 2 can fire.  Pins: the true condition number of the non-zero spectrum
    is > 1/eps (so 6 is the right answer), and scipy's LSQR stops with the same code at the same iteration."""
    rng = np.random.default_rng(16)
    k1, k2 = int(rng.integers(1, 8)), int(rng.integers(2, 12))
    k = k1 + k2
    m = k + int(rng.integers(1, 10))
    U, _ = np.linalg.qr(rng.standard_normal((m, k)))
    V, _ = np.linalg.qr(rng.standard_normal((24, k)))
    e = rng.uniform(15.5, 17.5)
    sig = np.concatenate([rng.uniform(0.5, 1, k1), 10 ** (-e) * rng.uniform(0.5, 2, k2)])
    A = U @ np.diag(sig) @ V.T
    b = rng.standard_normal(m)
    assert (k1, k2, m) == (4, 7, 19) and sig.max() / sig.min() > 1.0 / np.finfo(float).eps
    r = _dense24(A).lsqr(b, 200, 0.0, 0.0)
    rs = spla.lsqr(A, b, atol=0.0, btol=0.0, conlim=0.0, iter_lim=200)
    assert r.istop == 6 == rs[1]
    assert r.itn == rs[2]
    assert 1.0 + 1.0 / r.acond <= 1.0
    assert abs(r.acond - rs[6]) <= 1e-2 * rs[6]


def test_se_scale_when_m_not_greater_than_n():
    """m_tot <= n (the other branch): se = sqrt(var) * rnorm without the sqrt(m - n)
    divisor.  Pin: the Krylov closed form for var and the true residual of the dense Krylov solution."""
    rng = np.random.default_rng(5)
    A = rng.standard_normal((10, 24))
    b = rng.standard_normal(10)
    S = _dense24(A)
    assert S.m_tot <= S.n
    B, V, beta = _golub_kahan_reorth(A, b, 6)
    for k in (1, 3, 6):
        Bk, Vk = B[:k + 1, :k], V[:, :k]
        e1 = np.zeros(k + 1)
        e1[0] = beta
        zk = Vk @ np.linalg.lstsq(Bk, e1, rcond=None)[0]
        var_ref = np.diag(Vk @ np.linalg.inv(Bk.T @ Bk) @ Vk.T)
        rk = S.lsqr(b, k, 0.0, 0.0)
        assert (rk.istop, rk.itn) == (7, k)
        np.testing.assert_allclose(rk.se, np.sqrt(var_ref) * np.linalg.norm(b - A @ zk), rtol=1e-9)


# ----------------------------------------------------------------------------- OpenMP restatement (bench only)
@pytest.mark.parametrize("threads", [1, 3, 8])
def test_omp_restatement_matches_the_oracle(threads):
    """oracle/gsr_oracle_omp.c (PAPER.md:150 threading; used only for bench.py's all-core cpu_baseline) against
    the parity oracle: aprods within 1e-12 * sum|terms|, LSQR x within 1e-10 after 30 iterations."""
    cfg = synth.SynthConfig("omp", 700, 400, 90, obs_powerlaw=(2.0, 12, 60), n_con=7, con_nnz=30, seed=3)   # m > n, well posed
    S, d = oracle_system(cfg)
    b = make_b(S, d)
    R = oracle.OmpRunner(S, threads)
    assert R.threads == threads
    rng = np.random.default_rng(0)
    x, y = rng.standard_normal(S.n), rng.standard_normal(S.m_tot)
    y1, ab = S.aprod1(x, y, want_abs=True)
    assert np.all(np.abs(R.aprod1(x, y) - y1) <= 1e-12 * ab)
    x1, ab = S.aprod2(y, x, want_abs=True)
    assert np.all(np.abs(R.aprod2(y, x) - x1) <= 1e-12 * ab)
    S.precondition()
    r1, r2 = S.lsqr(b, 30, 0.0, 0.0), R.lsqr(b, 30, 0.0, 0.0)
    assert (r1.istop, r1.itn) == (r2.istop, r2.itn) == (7, 30)
    assert np.linalg.norm(r1.x - r2.x) <= 1e-10 * np.linalg.norm(r1.x)
    assert np.linalg.norm(r1.se - r2.se) <= 1e-9 * np.linalg.norm(r1.se)
    assert abs(r1.rnorm - r2.rnorm) <= 1e-10 * r1.rnorm


# ----------------------------------------------------------------------------- N_Glob != 1
@pytest.mark.parametrize("n_glob", [0, 2, 5])
def test_global_section_of_any_width(n_glob):
    """The paper's layout has N_Glob = 1 but it also ran 5 global parameters and allows none
    (PAPER.md:78): row width 23 + n_glob, global columns at the end of x.  Pins: the structure (every row touches
    every global column exactly once, in stored order), dense numpy products, adjoint identity, unit columns after
    preconditioning, and the least-squares solution from numpy."""
    cfg = dataclasses.replace(synth.mini(seed=11, n_stars=6, obs=14, n_dof_att=7, n_instr=6), n_glob=n_glob)
    S, d = oracle_system(cfg)
    assert S.V.shape == (84, 23 + n_glob) and S.n == 30 + 21 + 6 + n_glob
    for i in (0, 17, 83):
        assert [S.col(i, 23 + g) for g in range(n_glob)] == [S.n - n_glob + g for g in range(n_glob)]
        assert S.col(i, 22) == 30 + 21 + d["instrCol"][i, 5]
    A = dense(S)
    rng = np.random.default_rng(n_glob)
    x, y = rng.standard_normal(S.n), rng.standard_normal(S.m_tot)
    y1, ab = S.aprod1(x, y, want_abs=True)
    assert np.all(np.abs(y1 - (y + A @ x)) <= 1e-14 * ab)
    x1, ab = S.aprod2(y, x, want_abs=True)
    assert np.all(np.abs(x1 - (x + A.T @ y)) <= 1e-14 * ab)
    assert abs(np.dot(A @ x, y) - np.dot(x, S.aprod2(y, np.zeros(S.n)))) <= 1e-12 * np.linalg.norm(A @ x) * np.linalg.norm(y)
    b = make_b(S, d)
    p = S.precondition()
    np.testing.assert_allclose(np.linalg.norm(dense(S), axis=0), 1.0, rtol=1e-14)
    np.testing.assert_allclose(p, 1.0 / np.linalg.norm(A, axis=0), rtol=1e-14)
    r = S.lsqr(b, 500, 1e-15, 1e-15)
    xls = np.linalg.lstsq(A, b, rcond=None)[0]
    assert np.linalg.norm(r.x - xls) <= 1e-9 * np.linalg.norm(xls)
    if n_glob:   # the OpenMP restatement follows
        R = oracle.OmpRunner(S, 3)
        assert np.linalg.norm(R.lsqr(b, 500, 1e-15, 1e-15).x - r.x) <= 1e-9 * np.linalg.norm(r.x)


# ----------------------------------------------------------------------------- section widths other than 5/12/6/1 (NEXT-4)
def test_hand_worked_variant_fixture():
    """General column map (PAPER.md:78 widths; Alg. 2 index expressions) on a hand-worked 2/12/3/2 system
    (tests/golden/hand_variant.txt): columns, aprod1 and aprod2 values derived by hand."""
    rows, kv = [], {}
    for line in open(os.path.join(GOLD, "hand_variant.txt")):
        line = line.split("#")[0].strip()
        if not line:
            continue
        tok = line.split()
        if tok[0] == "row":
            a, b_, c = line[3:].split("|")
            ia, iatt = map(int, a.split())
            rows.append((ia, iatt, list(map(int, b_.split())), c.strip()))
        else:
            kv[tok[0]] = [float(t) for t in tok[1:]]
    w = {k: int(kv[k][0]) for k in ("n_astro_par", "n_att_par", "n_instr_par", "n_glob", "n_stars", "n_dof_att", "n_instr")}
    npar = w["n_astro_par"] + w["n_att_par"] + w["n_instr_par"] + w["n_glob"]
    assert npar == 19
    rule = {"ones": lambda k: 1.0, "kplus1": lambda k: k + 1.0}
    V = np.array([[rule[r[3]](k) for k in range(npar)] for r in rows])
    S = oracle.OracleSystem(w["n_stars"], w["n_dof_att"], w["n_instr"], V, [r[0] for r in rows], [r[1] for r in rows],
                            [r[2] for r in rows], n_glob=w["n_glob"], n_astro_par=w["n_astro_par"],
                            n_att_par=w["n_att_par"], n_instr_par=w["n_instr_par"])
    assert S.n == 25
    assert [S.col(1, k) for k in range(npar)] == [int(c) for c in kv["cols1"]]
    y, ab = S.aprod1(np.arange(1, 26, dtype=np.float64), np.array(kv["aprod1_yin"]), want_abs=True)
    assert y.tolist() == kv["aprod1_yout"]
    assert ab.tolist() == [100 + 253, 200 + 3407]      # all terms positive
    assert S.aprod2(np.array(kv["aprod2_y"]), np.zeros(25)).tolist() == kv["aprod2_xout"]


VARIANTS = [   # (n_astro_par, n_att_par, n_instr_par, n_glob): PAPER.md:78 ranges and the section subsets of PAPER.md:263
    (0, 12, 6, 0),    # attitude + instrumental only (the paper's 40 and 300 GB datasets)
    (5, 0, 0, 0),     # astrometric only (the 100 GB dataset)
    (5, 12, 6, 0),    # astrometric + attitude + instrumental, no global part (the 350 GB dataset)
    (3, 12, 4, 2),    # fewer astrometric / instrumental coefficients, two global parameters
    (2, 0, 1, 5),     # no attitude part, five global parameters
]


@pytest.mark.parametrize("widths", VARIANTS)
def test_section_width_variants(widths):
    """Every layout the paper allows reduces to the same definition with other widths.  Pins: structure of each row
    (block-diagonal astro part of N_Astro columns, 3 x 4 attitude columns N_DFA apart, instrument columns inside their
    range, every global column once), dense numpy products with their |terms| bounds, adjoint identity, unit columns
    after preconditioning, numpy's least-squares solution."""
    na, nt, ni, ng = widths
    cfg = dataclasses.replace(synth.mini(seed=5, n_stars=7, obs=16, n_dof_att=9, n_instr=7), n_glob=ng, n_astro_par=na,
                              n_att_par=nt, n_instr_par=ni)
    S, d = oracle_system(cfg)
    m, ns, nd = S.m, cfg.n_stars, cfg.n_dof_att
    off_att = na * ns
    off_instr = off_att + (3 * nd if nt else 0)
    off_glob = off_instr + (cfg.n_instr if ni else 0)
    assert S.n == off_glob + ng == cfg.n and S.V.shape == (m, na + nt + ni + ng)
    A = dense(S)
    assert ((A[:m] != 0).sum(axis=1) == na + nt + ni + ng).all()
    star = np.repeat(np.arange(ns), 16)
    for i in range(m):
        nz = np.nonzero(A[i])[0]
        assert nz[:na].tolist() == list(range(na * star[i], na * star[i] + na))
        if nt:
            att = nz[na:na + 12].reshape(3, 4)
            assert (np.diff(att, axis=1) == 1).all() and (np.diff(att[:, 0]) == nd).all()
            assert off_att <= att[0, 0] and att[0, 3] < off_att + nd
            assert att[0, 0] - off_att == d["matrixIndexAtt"][i]
        if ni:
            ins = nz[na + nt:na + nt + ni]
            assert sorted(ins - off_instr) == sorted(d["instrCol"][i].tolist())
        assert nz[na + nt + ni:].tolist() == list(range(off_glob, off_glob + ng))
        # stored order: coefficient k of the row sits in the k-th column of the map, with the stored value
        for k in range(S.n_par):
            assert A[i, S.col(i, k)] == S.V[i, k]
    rng = np.random.default_rng(sum(widths))
    x, y = rng.standard_normal(S.n), rng.standard_normal(S.m_tot)
    y1, ab = S.aprod1(x, y, want_abs=True)
    np.testing.assert_allclose(ab, np.abs(y) + np.abs(A) @ np.abs(x), rtol=1e-13)
    assert np.all(np.abs(y1 - (y + A @ x)) <= 1e-14 * ab)
    x1, ab = S.aprod2(y, x, want_abs=True)
    np.testing.assert_allclose(ab, np.abs(x) + np.abs(A).T @ np.abs(y), rtol=1e-13)
    assert np.all(np.abs(x1 - (x + A.T @ y)) <= 1e-14 * ab)
    assert abs(np.dot(A @ x, y) - np.dot(x, S.aprod2(y, np.zeros(S.n)))) <= 1e-12 * np.linalg.norm(A @ x) * np.linalg.norm(y)
    b = make_b(S, d)
    p = S.precondition()
    np.testing.assert_allclose(np.linalg.norm(dense(S), axis=0), 1.0, rtol=1e-14)
    np.testing.assert_allclose(p, 1.0 / np.linalg.norm(A, axis=0), rtol=1e-14)
    r = S.lsqr(b, 800, 1e-15, 1e-15)
    xls = np.linalg.lstsq(A, b, rcond=None)[0]
    assert np.linalg.norm(r.x - xls) <= 1e-9 * np.linalg.norm(xls)
