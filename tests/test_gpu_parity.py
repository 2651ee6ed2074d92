"""GPU parity: the CUDA path (through the C ABI) against the CPU oracle on the same seeded inputs.

Tolerances (BASELINE north_star): index/layout arrays bit-exact; every aprod output element within
1e-12 * sum|terms|; LSQR x after a fixed iteration count within 1e-9 relative L2, same istop,
itn within +-2.
"""
import dataclasses

import numpy as np
import pytest
import torch

import oracle
from helpers import make_b, np_inputs, oracle_system
from paper_2308_00778_b200 import synth

pytestmark = pytest.mark.gpu

APROD_TOL = 1e-12
X_TOL = 1e-9
P_TOL = 5e-14     # preconditioner factors / scaled coefficients (see test_precondition_parity)
SE_TOL = 1e-8     # standard errors: sqrt of a sum of squares of d_k = w_k / rho_k, each carrying x's 1e-9
X_TOL_CONVERGED = 1e-8   # x of a run that stops on its own: the two sides may stop up to 2 iterations apart (itn +-2 is
                         # the north-star bar) at the rounding floor, where one more iteration still moves x by ~1e-9 |x|


def gsr_mod():
    from paper_2308_00778_b200 import gsr
    return gsr


def dev(a):
    return torch.from_numpy(np.ascontiguousarray(a)).cuda()


def make_gpu(S, d, b, upload_constraints=True, flags=0):
    gsr = gsr_mod()
    G = gsr.Gsr(S.m, S.n_stars, S.n_dof_att, S.n_instr, S.n_con, len(S.con_col), flags=flags, n_glob=S.n_glob,
                n_astro_par=S.n_astro_par, n_att_par=S.n_att_par, n_instr_par=S.n_instr_par)
    # the index array of a section the layout does not have is not passed at all
    G.gsr_upload(np.ascontiguousarray(d["values"]),
                 np.ascontiguousarray(d["matrixIndexAstro"]) if S.n_astro_par else None,
                 np.ascontiguousarray(d["matrixIndexAtt"]) if S.n_att_par else None,
                 np.ascontiguousarray(d["instrCol"]) if S.n_instr_par else None, b)
    if S.n_con and upload_constraints:
        G.gsr_upload_constraints(S.con_rowptr, S.con_col, S.con_val)
    return G


def subset(d, keep):
    """Keep the rows of a generated system selected by the boolean mask `keep`."""
    out = dict(d)
    for k in ("values", "matrixIndexAstro", "matrixIndexAtt", "instrCol", "noise"):
        out[k] = np.ascontiguousarray(d[k][keep])
    return out


def check_aprods(S, G, seed=0):
    rng = np.random.default_rng(seed)
    x = rng.standard_normal(S.n)
    y = rng.standard_normal(S.m_tot)
    y1 = G.gsr_aprod1(dev(x), dev(y)).cpu().numpy()
    y1o, ab = S.aprod1(x, y, want_abs=True)
    assert np.all(np.abs(y1 - y1o) <= APROD_TOL * ab + 1e-300), np.max(np.abs(y1 - y1o) / (ab + 1e-300))
    x2 = G.gsr_aprod2(dev(y), dev(x)).cpu().numpy()
    x2o, ab2 = S.aprod2(y, x, want_abs=True)
    assert np.all(np.abs(x2 - x2o) <= APROD_TOL * ab2 + 1e-300), np.max(np.abs(x2 - x2o) / (ab2 + 1e-300))
    return x, y


CASES = {
    "mini": dict(cfg=synth.mini(seed=1)),
    "mini_con": dict(cfg=synth.mini(seed=2, n_stars=40, obs=9, n_dof_att=30, n_instr=16, n_con=5, con_nnz=20)),
    "ragged_tail": dict(cfg=synth.mini(seed=3, n_stars=37, obs=23, n_dof_att=64, n_instr=10)),        # 851 rows
    "one_row_stars": dict(cfg=synth.mini(seed=4, n_stars=300, obs=1, n_dof_att=40, n_instr=9)),       # every tile full of heads
    "one_star": dict(cfg=synth.mini(seed=5, n_stars=1, obs=1000, n_dof_att=200, n_instr=6)),          # one segment over 32 tiles
    "tiny_rows": dict(cfg=synth.mini(seed=6, n_stars=3, obs=5, n_dof_att=4, n_instr=6)),              # m < 32, N_DFA = 4
    # Skewed-like: power-law rows per star, bursty attitude times, Zipf instrument columns.
    # kmin = 1 (many stars cut to 1-2 rows; rank deficient, aprod parity only) and kmin = 8 (well posed).
    "powerlaw_short": dict(cfg=synth.SynthConfig("pl1", 400, 300, 50, obs_powerlaw=(2.0, 1, 200),
                                                 att_bursts=(5, 1e-2, 0.9), instr_zipf=1.1, seed=7)),
    "powerlaw": dict(cfg=synth.SynthConfig("pl8", 400, 300, 50, obs_powerlaw=(2.0, 8, 200),
                                           att_bursts=(5, 1e-2, 0.9), instr_zipf=1.1, seed=7)),
    # Zipf(1.1) over 2,000 columns: the hottest column holds ~300x the mean, which switches aprod2 to the
    # variant that pre-sums equal columns inside a warp (MATCH)
    "zipf_hot": dict(cfg=synth.SynthConfig("zipf", 300, 200, 2_000, obs_per_star=30, instr_zipf=1.1, seed=9)),
    # more than 65,536 instrument columns: the device keeps 4-byte columns (2-byte ones otherwise)
    "wide_instr": dict(cfg=synth.SynthConfig("wide", 200, 150, 70_000, obs_per_star=40, seed=12)),
    "zipf_con": dict(cfg=synth.SynthConfig("zipfc", 300, 200, 2_000, obs_per_star=30, instr_zipf=1.1, n_con=6,
                                           con_nnz=40, seed=10)),
}


@pytest.mark.parametrize("name", list(CASES))
def test_aprod_parity_and_layout(name):
    cfg = CASES[name]["cfg"]
    S, d = oracle_system(cfg)
    b = make_b(S, d)
    with make_gpu(S, d, b) as G:
        assert G.n == S.n and G.m_tot == S.m_tot
        assert bool(G.gsr_path_info() & gsr_mod().GSR_PATH_IC16) == (cfg.n_instr <= 65536)
        rp = G.gsr_get_star_rowptr().cpu().numpy()
        assert np.array_equal(rp, d["rowptr"])                                   # generator's own
        assert np.array_equal(rp, np.searchsorted(S.ia, 5 * np.arange(S.n_stars + 1), side="left"))
        check_aprods(S, G)


def test_stars_without_rows_and_empty_system():
    cfg = synth.mini(seed=8, n_stars=50, obs=20, n_dof_att=30, n_instr=8)
    d = np_inputs(cfg)
    star = d["matrixIndexAstro"] // 5
    keep = ~np.isin(star, [0, 7, 8, 9, 30, 49])      # first, a run, one in the middle, last
    ds = subset(d, keep)
    S = oracle.OracleSystem(cfg.n_stars, cfg.n_dof_att, cfg.n_instr, ds["values"], ds["matrixIndexAstro"],
                            ds["matrixIndexAtt"], ds["instrCol"])
    b = S.aprod1(d["x_true"], ds["noise"])
    with make_gpu(S, ds, b) as G:
        rp = G.gsr_get_star_rowptr().cpu().numpy()
        assert np.array_equal(rp, np.searchsorted(S.ia, 5 * np.arange(S.n_stars + 1), side="left"))
        check_aprods(S, G)
        G.gsr_precondition()
        p = G.gsr_get_colscale().cpu().numpy()
        po = S.precondition()
        assert np.all(p[po == 1.0] == 1.0)           # empty columns: p = 1 (reading R2)
        np.testing.assert_allclose(p, po, rtol=P_TOL, atol=0)
    # m = 0
    gsr = gsr_mod()
    e = np.zeros((0, 24))
    with gsr.Gsr(0, 4, 8, 8) as G:
        G.gsr_upload(e, np.zeros(0, np.int64), np.zeros(0, np.int64), np.zeros((0, 6), np.int32), np.zeros(0))
        x = torch.ones(G.n, dtype=torch.float64, device="cuda")
        y = torch.zeros(0, dtype=torch.float64, device="cuda")
        G.gsr_aprod2(y, x)
        assert torch.all(x == 1.0)
        r = G.gsr_lsqr(5, 0.0, 0.0)
        assert r.istop == 0 and r.itn == 0 and torch.all(r.x == 0)


def test_tiny_config_aprod_parity():
    cfg = synth.tiny()
    S, d = oracle_system(cfg)
    b = make_b(S, d)
    with make_gpu(S, d, b) as G:
        check_aprods(S, G)


def test_astro_and_gamma_are_bit_reproducible():
    cfg = synth.tiny()
    S, d = oracle_system(cfg)
    b = make_b(S, d)
    rng = np.random.default_rng(5)
    y = dev(rng.standard_normal(S.m))
    with make_gpu(S, d, b) as G:
        outs = []
        for _ in range(3):
            x = torch.zeros(S.n, dtype=torch.float64, device="cuda")
            outs.append(G.gsr_aprod2(y, x).cpu().numpy())
        na = 5 * cfg.n_stars
        for o in outs[1:]:
            assert np.array_equal(o[:na], outs[0][:na])
            assert o[-1] == outs[0][-1]
    # with the column-ordered instrument copy (opt-in) that section is summed without atomics, in a fixed order too
    with make_gpu(S, d, b, flags=gsr_mod().GSR_FLAG_INS_COPY) as G:
        assert G.gsr_path_info() & gsr_mod().GSR_PATH_INS_COPY
        outs = [G.gsr_aprod2(y, torch.zeros(S.n, dtype=torch.float64, device="cuda")).cpu().numpy() for _ in range(3)]
        oi = 5 * cfg.n_stars + 3 * cfg.n_dof_att
        for o in outs[1:]:
            assert np.array_equal(o[:na], outs[0][:na])
            assert np.array_equal(o[oi:], outs[0][oi:])


@pytest.mark.parametrize("name", ["mini_con", "ragged_tail", "powerlaw"])
def test_precondition_parity(name):
    cfg = CASES[name]["cfg"]
    S, d = oracle_system(cfg)
    b = make_b(S, d)
    with make_gpu(S, d, b) as G:
        G.gsr_precondition()
        p = G.gsr_get_colscale().cpu().numpy()
        po = S.precondition()
        # column sums of squares are positive sums taken in a different order on the two sides:
        # relative difference <= N_col * eps (N_col ~ 1e2..1e3 terms here), halved by the sqrt
        np.testing.assert_allclose(p, po, rtol=P_TOL, atol=0)
        V, cv = G.gsr_get_values()
        # A' = fl(A * p): inherits p's relative difference plus one rounding
        np.testing.assert_allclose(V.cpu().numpy(), S.V, rtol=P_TOL, atol=0)
        if S.n_con:
            np.testing.assert_allclose(cv.cpu().numpy(), S.con_val, rtol=P_TOL, atol=0)
        with pytest.raises(gsr_mod().GsrError) as e:
            G.gsr_precondition()
        assert e.value.code == gsr_mod().GSR_ESTATE
        check_aprods_scaled(S, G)


def check_aprods_scaled(S, G):
    """aprods on the preconditioned matrices: the two stored matrices differ by rounding of p,
    so the bound gets the P_TOL relative slack of the stored values on top of 1e-12."""
    rng = np.random.default_rng(1)
    x = rng.standard_normal(S.n)
    y = rng.standard_normal(S.m_tot)
    y1 = G.gsr_aprod1(dev(x), dev(y)).cpu().numpy()
    y1o, ab = S.aprod1(x, y, want_abs=True)
    assert np.all(np.abs(y1 - y1o) <= (APROD_TOL + P_TOL) * ab)
    x2 = G.gsr_aprod2(dev(y), dev(x)).cpu().numpy()
    x2o, ab2 = S.aprod2(y, x, want_abs=True)
    assert np.all(np.abs(x2 - x2o) <= (APROD_TOL + P_TOL) * ab2)


def lsqr_both(cfg, itnlim, atol, btol, conlim=0.0, precond=True, noise=True):
    S, d = oracle_system(cfg)
    if not noise:
        d["noise"] = np.zeros_like(d["noise"])
    b = make_b(S, d)
    G = make_gpu(S, d, b)
    if precond:
        G.gsr_precondition()
        S.precondition()
    r = G.gsr_lsqr(itnlim, atol, btol, conlim)
    ro = S.lsqr(b, itnlim, atol, btol, conlim, want_trace=True)
    return S, d, G, r, ro


def rel(a, b):
    return np.linalg.norm(a - b) / max(np.linalg.norm(b), 1e-300)


@pytest.mark.parametrize("name,itn", [("mini", 30), ("mini_con", 25), ("ragged_tail", 40), ("powerlaw", 40),
                                      ("zipf_hot", 30), ("zipf_con", 30), ("wide_instr", 20)])
def test_lsqr_fixed_iterations_small(name, itn):
    S, d, G, r, ro = lsqr_both(CASES[name]["cfg"], itn, 0.0, 0.0)
    with G:
        if name.startswith("zipf"):      # the variant that pre-sums equal instrument columns inside a warp was chosen
            assert G.gsr_path_info() & gsr_mod().GSR_PATH_INSTR_MATCH
        assert (r.istop, r.itn) == (ro.istop, ro.itn) == (7, itn)
        assert rel(r.x.cpu().numpy(), ro.x) <= X_TOL
        assert rel(r.se.cpu().numpy(), ro.se) <= SE_TOL
        for a, bb in ((r.rnorm, ro.rnorm), (r.anorm, ro.anorm), (r.acond, ro.acond), (r.xnorm, ro.xnorm)):
            assert abs(a - bb) <= 1e-9 * abs(bb)
        assert abs(r.arnorm - ro.arnorm) <= 1e-9 * ro.anorm * ro.rnorm + 1e-9 * abs(ro.arnorm)
        tr = G.gsr_get_trace()
        assert tr.shape == (itn, 5)
        np.testing.assert_allclose(tr[:, 0], ro.trace[:, 0], rtol=1e-9)
        np.testing.assert_allclose(tr[:, 2], ro.trace[:, 2], rtol=1e-9)


def test_lsqr_tiny_config_fixed_40_iterations():
    """BASELINE configs[0], x parity at a fixed iteration count before the rounding floor
    (reading R19): 40 iterations, atol = btol = 0, istop 7 on both sides."""
    S, d, G, r, ro = lsqr_both(synth.tiny(), 40, 0.0, 0.0)
    with G:
        assert (r.istop, r.itn) == (ro.istop, ro.itn) == (7, 40)
        assert rel(r.x.cpu().numpy(), ro.x) <= X_TOL
        assert rel(r.se.cpu().numpy(), ro.se) <= SE_TOL
        assert rel(r.x.cpu().numpy(), d["x_true"]) <= 1e-2


def test_lsqr_tiny_config_100_iterations():
    """BASELINE configs[0] as stated: itnlim 100.  The preconditioned Tiny system reaches the
    rounding floor (1 + test2 <= 1, istop 5) near iteration 50 on both sides: same istop,
    itn within +-2, x within 1e-9."""
    S, d, G, r, ro = lsqr_both(synth.tiny(), 100, 0.0, 0.0)
    with G:
        assert r.istop == ro.istop
        assert abs(r.itn - ro.itn) <= 2, (r.itn, ro.itn)
        assert rel(r.x.cpu().numpy(), ro.x) <= X_TOL
        assert rel(r.se.cpu().numpy(), ro.se) <= 1e-7


def test_lsqr_stop_tests_match():
    # atol = btol = 1e-14 (BASELINE Tiny): same istop, itn within +-2
    S, d, G, r, ro = lsqr_both(synth.tiny(), 400, 1e-14, 1e-14)
    with G:
        assert r.istop == ro.istop and r.istop != 7
        assert abs(r.itn - ro.itn) <= 2, (r.itn, ro.itn)
        assert rel(r.x.cpu().numpy(), ro.x) <= X_TOL_CONVERGED
    # loose tolerances stop early on test 2; conlim test 3; consistent system test 1
    for kw in (dict(atol=1e-6, btol=1e-6), dict(atol=0.0, btol=0.0, conlim=5.0),
               dict(atol=1e-10, btol=1e-10, noise=False)):
        noise = kw.pop("noise", True)
        S, d, G, r, ro = lsqr_both(CASES["ragged_tail"]["cfg"], 300, kw.get("atol"), kw.get("btol"),
                                   kw.get("conlim", 0.0), noise=noise)
        with G:
            assert r.istop == ro.istop and r.istop in (1, 2, 3), (kw, r.istop, ro.istop)
            assert abs(r.itn - ro.itn) <= 2


def test_lsqr_unpreconditioned_and_host_output():
    cfg = CASES["mini"]["cfg"]
    S, d = oracle_system(cfg)
    b = make_b(S, d)
    with make_gpu(S, d, b) as G:
        r = G.gsr_lsqr(20, 0.0, 0.0, host_out=True)
        ro = S.lsqr(b, 20, 0.0, 0.0)
        assert not r.x.is_cuda
        assert rel(r.x.numpy(), ro.x) <= X_TOL
        # a second solve on the same handle reuses the captured graph and gives the same answer
        r2 = G.gsr_lsqr(20, 0.0, 0.0)
        assert rel(r2.x.cpu().numpy(), ro.x) <= X_TOL
        assert r2.kernel_launches > 0 and r2.loop_ms > 0


@pytest.mark.parametrize("name", ["mini_con", "powerlaw"])
def test_covariances_of_couples(name):
    """gsr_set_cov_pairs / gsr_get_cov (Alg. 1 l.26-27; R26) against the oracle's
    gsr_oracle_lsqr_cov: couples drawn over all sections plus some (i, i); tolerance SE_TOL relative to se_i se_j (the
    Cauchy-Schwarz scale of a covariance); fused and two-product iteration; cov(i, i) = se_i^2; couples persist over
    solves and can be cleared; a couple outside [0, n) is GSR_EINDEX."""
    gsr = gsr_mod()
    cfg = CASES[name]["cfg"]
    S, d = oracle_system(cfg)
    b = make_b(S, d)
    rng = np.random.default_rng(12)
    pi = np.concatenate([rng.integers(0, S.n, 500), np.arange(0, S.n, max(1, S.n // 40))]).astype(np.int64)
    pj = np.concatenate([rng.integers(0, S.n, 500), np.arange(0, S.n, max(1, S.n // 40))]).astype(np.int64)
    S.precondition()
    ro = S.lsqr(b, 20, 0.0, 0.0, pairs=(pi, pj))
    scale = ro.se[pi] * ro.se[pj]
    for flags in (0, gsr.GSR_FLAG_NO_FUSE):
        with make_gpu(S, {**d, "values": S.V}, b, flags=flags) as G:       # the preconditioned matrix: p = 1 on the device
            with pytest.raises(gsr.GsrError) as e:
                G.gsr_get_cov()
            assert e.value.code == gsr.GSR_ESTATE
            G.gsr_set_cov_pairs(pi, pj)
            for _ in range(2):                                              # the couples stay set; the sums start at zero
                r = G.gsr_lsqr(20, 0.0, 0.0)
                cov = G.gsr_get_cov().cpu().numpy() * S.p[pi] * S.p[pj]
                assert (r.istop, r.itn) == (ro.istop, ro.itn) == (7, 20)
                assert np.all(np.abs(cov - ro.cov) <= SE_TOL * scale), float(np.max(np.abs(cov - ro.cov) / scale))
                se = r.se.cpu().numpy() * S.p
                np.testing.assert_allclose(cov[500:], se[pi[500:]] ** 2, rtol=1e-12)
                assert rel(r.x.cpu().numpy() * S.p, ro.x) <= X_TOL
            bad = pj.copy()
            bad[7] = S.n
            with pytest.raises(gsr.GsrError) as e:
                G.gsr_set_cov_pairs(pi, bad)
            assert e.value.code == gsr.GSR_EINDEX and "couple 7" in str(e.value)
            G.gsr_set_cov_pairs(None, None)
            r = G.gsr_lsqr(20, 0.0, 0.0)
            assert rel(r.x.cpu().numpy() * S.p, ro.x) <= X_TOL
            with pytest.raises(gsr.GsrError):
                G.gsr_get_cov()
    # with the device's own preconditioner: cov carries p_i p_j
    S2, _ = oracle_system(cfg)
    with make_gpu(S2, d, b) as G:
        G.gsr_precondition()
        G.gsr_set_cov_pairs(dev(pi), dev(pj))                               # device arrays
        G.gsr_lsqr(20, 0.0, 0.0)
        cov = G.gsr_get_cov().cpu().numpy()
        assert np.all(np.abs(cov - ro.cov) <= SE_TOL * scale)


def test_b_zero_gives_istop0():
    cfg = CASES["mini"]["cfg"]
    S, d = oracle_system(cfg)
    with make_gpu(S, d, np.zeros(S.m_tot)) as G:
        r = G.gsr_lsqr(10, 1e-10, 1e-10)
        assert r.istop == 0 and r.itn == 0 and torch.all(r.x == 0)


def test_index_validation():
    gsr = gsr_mod()
    cfg = CASES["mini"]["cfg"]
    S, d = oracle_system(cfg)
    b = make_b(S, d)
    for key, row, val in (("matrixIndexAstro", 17, 3), ("matrixIndexAtt", 40, cfg.n_dof_att - 3),
                          ("instrCol", 100, cfg.n_instr), ("matrixIndexAstro", 5, 5 * cfg.n_stars),
                          ("instrCol", 33, 65536 + 3), ("instrCol", 7, -1)):      # would alias a valid 2-byte column
        bad = {k: np.array(v, copy=True) for k, v in d.items()}
        if key == "instrCol":
            bad[key][row, 2] = val
        else:
            bad[key][row] = val
        G = gsr.Gsr(S.m, S.n_stars, S.n_dof_att, S.n_instr)
        with G:
            with pytest.raises(gsr.GsrError) as e:
                G.gsr_upload(bad["values"], bad["matrixIndexAstro"], bad["matrixIndexAtt"], bad["instrCol"], b)
            assert e.value.code == gsr.GSR_EINDEX
            assert G.gsr_bad_row() in (row, row + 1)
            with pytest.raises(gsr.GsrError) as e2:     # nothing usable was uploaded
                G.gsr_precondition()
            assert e2.value.code == gsr.GSR_ESTATE
    with pytest.raises(gsr.GsrError) as e:
        gsr.Gsr(10, 2, 3, 8)                             # N_DFA < 4
    assert e.value.code == gsr.GSR_EINVAL


def test_chunked_device_upload_equals_whole_upload():
    cfg = CASES["ragged_tail"]["cfg"]
    S, d = oracle_system(cfg)
    b = make_b(S, d)
    gsr = gsr_mod()
    with gsr.Gsr(S.m, S.n_stars, S.n_dof_att, S.n_instr) as G:
        step = 300
        for r0 in range(0, S.m, step):
            r1 = min(r0 + step, S.m)
            G.gsr_upload_rows(r0, r1 - r0, dev(d["values"][r0:r1]), dev(d["matrixIndexAstro"][r0:r1]),
                              dev(d["matrixIndexAtt"][r0:r1]), dev(d["instrCol"][r0:r1]), dev(b[r0:r1]))
        G.gsr_upload_finish()
        check_aprods(S, G)


def test_upload_state_partial_reupload_and_abandoned_upload():
    """gsr_upload_finish needs every row since the last finish (the per-row star scratch is rebuilt per upload): a
    partial re-upload is GSR_ESTATE, not a row pointer derived from stale memory.  And a chunk with a column that does
    not fit 2 bytes, sent in an upload that is then abandoned, leaves nothing behind once its rows come again."""
    cfg = CASES["ragged_tail"]["cfg"]
    S, d = oracle_system(cfg)
    b = make_b(S, d)
    gsr = gsr_mod()
    half = S.m // 2

    def send(G, r0, r1, instr=None):
        G.gsr_upload_rows(r0, r1 - r0, d["values"][r0:r1], d["matrixIndexAstro"][r0:r1], d["matrixIndexAtt"][r0:r1],
                          np.ascontiguousarray((d["instrCol"] if instr is None else instr)[r0:r1]), b[r0:r1])

    with gsr.Gsr(S.m, S.n_stars, S.n_dof_att, S.n_instr) as G:
        with pytest.raises(gsr.GsrError) as e:               # nothing sent at all
            G.gsr_upload_finish()
        assert e.value.code == gsr.GSR_ESTATE
        send(G, 0, S.m)
        G.gsr_upload_finish()
        check_aprods(S, G)
        send(G, 0, half)                                     # partial re-upload
        with pytest.raises(gsr.GsrError) as e:
            G.gsr_upload_finish()
        assert e.value.code == gsr.GSR_ESTATE and str(half) in str(e.value)
        with pytest.raises(gsr.GsrError) as e:               # and the handle is not usable in between
            G.gsr_aprod1(dev(np.zeros(S.n)), dev(np.zeros(S.m)))
        assert e.value.code == gsr.GSR_ESTATE
        send(G, half, S.m)                                   # the rest, out of order with an overlap
        send(G, half - 7, half + 9)
        G.gsr_upload_finish()
        check_aprods(S, G, seed=3)
        # abandoned upload with a bad 2-byte column, then a clean one in another chunking
        bad = np.array(d["instrCol"], copy=True)
        bad[40, 1] = 65536 + 2
        send(G, 0, 100, instr=bad)
        send(G, 0, 60)
        send(G, 60, S.m)
        G.gsr_upload_finish()
        check_aprods(S, G, seed=4)
        # the same bad chunk, not replaced: reported with its row
        send(G, 100, S.m)
        send(G, 0, 100, instr=bad)
        with pytest.raises(gsr.GsrError) as e:
            G.gsr_upload_finish()
        assert e.value.code == gsr.GSR_EINDEX and G.gsr_bad_row() == 40
        send(G, 30, 50)                                      # after a failed finish the other rows are still there
        G.gsr_upload_finish()
        check_aprods(S, G, seed=5)


@pytest.mark.parametrize("ins_copy", [True, False])
def test_two_attitude_blocks_and_mixed_instrument_table(ins_copy):
    """2.2 M rows: more than one 2^21-row block of the block-time-ordered attitude copy, 269 row blocks of the
    column-ordered instrument copy (opt-in, the last one ragged), and 30,000 instrument columns: four column buckets for
    k_ins_scatter; without that copy more than the per-CTA shared-memory table holds, so both the ATOMS and the RED
    path run."""
    cfg = synth.SynthConfig("blocks2", 22_000, 4_000, 30_000, obs_per_star=100, seed=11)
    S, d = oracle_system(cfg)
    assert S.m > (1 << 21)
    b = make_b(S, d)
    with make_gpu(S, d, b, flags=gsr_mod().GSR_FLAG_INS_COPY if ins_copy else 0) as G:
        assert bool(G.gsr_path_info() & gsr_mod().GSR_PATH_INS_COPY) == ins_copy
        check_aprods(S, G)
        v, _ = G.gsr_get_values()
        assert np.array_equal(v.cpu().numpy(), d["values"])                     # layout round trip, bit-exact
        G.gsr_precondition()
        S.precondition()
        check_aprods(S, G, seed=1)
        r = G.gsr_lsqr(8, 0.0, 0.0)
        ro = S.lsqr(b, 8, 0.0, 0.0)
        assert r.istop == ro.istop == 7 and r.itn == ro.itn == 8
        xg = r.x.cpu().numpy()
        assert np.linalg.norm(xg - ro.x) <= X_TOL * np.linalg.norm(ro.x)


def stream_oracle_aprods(cfg, G, x, y, y1, x2, chunk_stars, threads=8, x_extra=None, ab_extra=None):
    """Chunk-streamed oracle over a system that exists only on the device: the rows of `chunk_stars`
    stars at a time are regenerated on the device (same seeded generator, same bytes as the upload), copied to the
    host and handed to oracle/gsr_oracle.c.  aprod1 is row-local: every row of y1 = A x is compared; aprod2
    accumulates across chunks (x_ref, and the bound sum|terms|, are sums of the chunks' contributions): every entry of
    x2 = A^T y is compared.  Chunks run on `threads` host threads (the oracle itself stays single-threaded C)."""
    from concurrent.futures import ThreadPoolExecutor
    dv = x.device
    rp = synth.star_rowptr(cfg, dv)
    xc = x.cpu().numpy()
    n = xc.shape[0]
    x_ref, ab_ref = np.zeros(n), np.zeros(n)
    worst1 = 0.0
    rows_checked = 0

    def work(P, r0, nr):
        So = oracle.OracleSystem(cfg.n_stars, cfg.n_dof_att, cfg.n_instr, P["values"], P["matrixIndexAstro"],
                                 P["matrixIndexAtt"], P["instrCol"])
        yo, ab = So.aprod1(xc, np.zeros(nr), want_abs=True)
        xo, ab2 = So.aprod2(P["y"], np.zeros(n), want_abs=True)
        return r0, nr, yo, ab, xo, ab2

    with ThreadPoolExecutor(threads) as pool:
        futs = []

        def drain(keep):
            nonlocal worst1, rows_checked
            while len(futs) > keep:
                r0, nr, yo, ab, xo, ab2 = futs.pop(0).result()
                yg = y1[r0:r0 + nr].cpu().numpy()
                err = np.abs(yg - yo) / (ab + 1e-300)
                assert np.all(err <= APROD_TOL), (r0, float(err.max()))
                worst1 = max(worst1, float(err.max()))
                np.add(x_ref, xo, out=x_ref)
                np.add(ab_ref, ab2, out=ab_ref)
                rows_checked += nr

        for s0 in range(0, cfg.n_stars, chunk_stars):
            part = synth.generate_rows(cfg, s0, min(s0 + chunk_stars, cfg.n_stars), dv, rp)
            r0, nr = part["row0"], part["values"].shape[0]
            P = {k: part[k].cpu().numpy() for k in ("values", "matrixIndexAstro", "matrixIndexAtt", "instrCol")}
            P["y"] = y[r0:r0 + nr].cpu().numpy()
            del part
            futs.append(pool.submit(work, P, r0, nr))
            drain(threads)
        drain(0)
    assert rows_checked == y1.shape[0]
    if x_extra is not None:     # contribution of rows the caller ran through the oracle itself (constraint rows)
        x_ref += x_extra
        ab_ref += ab_extra
    xg = x2.cpu().numpy()
    err2 = np.abs(xg - x_ref) / (ab_ref + 1e-300)
    return worst1, err2


def test_medium_full_size_every_element():
    """BASELINE configs[2] at full size (200 M rows) in the launch configuration bench.py times: EVERY one of the
    200,000,000 outputs of aprod1 and EVERY one of the 8,060,001 outputs of aprod2 (astro, attitude, instrument and
    gamma sections: the block-time-ordered copy over 96 blocks, the RED replicas, the per-CTA partials) against the
    chunk-streamed oracle at 1e-12 * sum|terms|; plus the adjoint identity over the whole system."""
    import bench
    gsr = gsr_mod()
    free, _ = torch.cuda.mem_get_info()
    if free < 90e9:
        pytest.skip("needs ~80 GB of free HBM")
    cfg = synth.medium()
    dv = torch.device("cuda", 0)
    m = int(synth.star_rowptr(cfg)[-1])
    with gsr.Gsr(m, cfg.n_stars, cfg.n_dof_att, cfg.n_instr) as G:
        bench.build_on_device(cfg, G, dv, torch, synth)
        info = G.gsr_path_info()
        assert info & gsr.GSR_PATH_ATT_COPY and info & gsr.GSR_PATH_FUSED and info & gsr.GSR_PATH_IC16
        g = torch.Generator(device="cuda").manual_seed(5)
        x = torch.randn(G.n, dtype=torch.float64, device=dv, generator=g)
        y = torch.randn(m, dtype=torch.float64, device=dv, generator=g)
        y1 = G.gsr_aprod1(x, torch.zeros(m, dtype=torch.float64, device=dv))
        x2 = G.gsr_aprod2(y, torch.zeros(G.n, dtype=torch.float64, device=dv))
        lhs, rhs = float(torch.dot(y1, y)), float(torch.dot(x, x2))
        scale = float(torch.linalg.norm(y1) * torch.linalg.norm(y))
        assert abs(lhs - rhs) <= 1e-11 * scale, (lhs, rhs, scale)
        worst1, err2 = stream_oracle_aprods(cfg, G, x, y, y1, x2, chunk_stars=10_000)
        na, nd = 5 * cfg.n_stars, cfg.n_dof_att
        sect = {"astro": err2[:na], "att": err2[na:na + 3 * nd], "instr": err2[na + 3 * nd:-1], "gamma": err2[-1:]}
        worst = {k: float(v.max()) for k, v in sect.items()}
        assert all(w <= APROD_TOL for w in worst.values()), worst
        print(f"medium every element: aprod1 worst {worst1:.2e}, aprod2 worst by section {worst} (x 1e-12 bound)")


def test_medium_lsqr_fused_path_vs_oracle():
    """BASELINE configs[2] at full size through gsr_lsqr on the path bench.py times (fused single pass, texture gathers,
    u kept in block-time order, 2-byte instrument columns; coefficient offsets beyond 2^32, 96 attitude blocks, most
    instrument adds outside the shared-memory table) and through the two-product form, against the oracle's LSQR on the
    same bytes: 3 iterations (a few LSQR iterations at Medium when the host has the RAM; the one-thread
    oracle needs ~45 s per iteration), Alg. 1 l.13-27.  b = A x_true + noise is formed by the oracle."""
    import psutil
    gsr = gsr_mod()
    torch.cuda.empty_cache()
    free, _ = torch.cuda.mem_get_info()
    if free < 90e9 or psutil.virtual_memory().available < 120e9:
        pytest.skip("needs ~80 GB of free HBM and ~100 GB of host RAM")
    cfg = synth.medium()
    dv = torch.device("cuda", 0)
    rp = synth.star_rowptr(cfg, dv)
    m = int(rp[-1])
    V = np.empty((m, 24))
    ia, iatt = np.empty(m, dtype=np.int64), np.empty(m, dtype=np.int64)
    ic = np.empty((m, 6), dtype=np.int32)
    noise = np.empty(m)
    for s0 in range(0, cfg.n_stars, 20_000):      # generated on the device (same seeded generator as the bench), kept on the host
        part = synth.generate_rows(cfg, s0, min(s0 + 20_000, cfg.n_stars), dv, rp)
        r0, nr = part["row0"], part["values"].shape[0]
        V[r0:r0 + nr] = part["values"].cpu().numpy()
        ia[r0:r0 + nr] = part["matrixIndexAstro"].cpu().numpy()
        iatt[r0:r0 + nr] = part["matrixIndexAtt"].cpu().numpy()
        ic[r0:r0 + nr] = part["instrCol"].cpu().numpy()
        noise[r0:r0 + nr] = part["noise"].cpu().numpy()
        del part
    torch.cuda.empty_cache()
    S = oracle.OracleSystem(cfg.n_stars, cfg.n_dof_att, cfg.n_instr, V, ia, iatt, ic)
    del V, ia, iatt, ic
    b = S.aprod1(synth.x_true(cfg, dv).cpu().numpy(), noise)
    got = {}
    for flags in (0, gsr.GSR_FLAG_NO_FUSE):
        with gsr.Gsr(m, cfg.n_stars, cfg.n_dof_att, cfg.n_instr, flags=flags) as G:
            G.gsr_upload(S.V, S.ia, S.iatt, S.ic, b)          # the unscaled bytes: S.precondition() comes later
            info = G.gsr_path_info()
            want = gsr.GSR_PATH_ATT_COPY | gsr.GSR_PATH_IC16 | (0 if flags else gsr.GSR_PATH_FUSED | gsr.GSR_PATH_TEX | gsr.GSR_PATH_UT)
            assert info & want == want and bool(info & gsr.GSR_PATH_FUSED) == (flags == 0), info
            G.gsr_precondition()
            p = G.gsr_get_colscale().cpu().numpy()
            r = G.gsr_lsqr(3, 0.0, 0.0)
            got[flags] = (p, r, r.x.cpu().numpy(), r.se.cpu().numpy(), G.gsr_get_trace())
        torch.cuda.empty_cache()
    # p_j = 1/sqrt(sum of squares of column j): positive sums taken in different orders on the two sides differ by at most
    # N_j * eps relatively (N_j = entries of the column), halved by the square root -- the derivation behind P_TOL, which
    # assumes N_j ~ 1e3.  Here N_j is 200 (astro), ~800 (attitude), ~20,000 (instrument) and 2e8 (gamma): per-column bound.
    na, nd = 5 * cfg.n_stars, cfg.n_dof_att
    cnt = np.empty(S.n)
    cnt[:na] = np.repeat(np.diff(rp.cpu().numpy()), 5)
    starts = np.bincount(S.iatt, minlength=nd).astype(np.float64)
    att = sum(np.concatenate([np.zeros(j), starts[:nd - j]]) for j in range(4))   # column c: rows with start in [c-3, c]
    cnt[na:na + 3 * nd] = np.tile(att, 3)
    cnt[na + 3 * nd:-1] = np.bincount(S.ic.reshape(-1), minlength=cfg.n_instr)
    cnt[-1] = m
    p_tol = np.maximum(P_TOL, 0.5 * cnt * np.finfo(np.float64).eps)
    S.precondition()
    ro = S.lsqr(b, 3, 0.0, 0.0, 0.0, True)
    assert (ro.istop, ro.itn) == (7, 3)
    report = {}
    for flags, (p, r, x, se, tr) in got.items():
        perr = np.abs(p - S.p) / S.p
        report[flags] = dict(stop=(r.istop, r.itn), p_worst=float((perr / p_tol).max()), p_max_rel=float(perr.max()),
                             p_argmax=int(perr.argmax()), x=rel(x, ro.x), se=rel(se, ro.se),
                             trace=float(np.max(np.abs(tr[:, (0, 2, 4)] / ro.trace[:, (0, 2, 4)] - 1.0))))
    print(f"medium lsqr vs oracle (flags -> figures): {report}")
    for flags, f in report.items():
        assert f["stop"] == (7, 3), (flags, f)
        assert f["p_worst"] <= 1.0, (flags, f)
        assert f["x"] <= X_TOL and f["se"] <= SE_TOL, (flags, f)
        assert f["trace"] <= 1e-9, (flags, f)                # rnorm, anorm, xnorm per iteration


def test_rows_unsorted_in_time_and_repeated_instrument_columns():
    """Inputs the header allows and the generator never makes (the instrument columns of a row follow no
    particular scheme; nothing orders a star's rows in time): the rows of every star shuffled, and 5 % of the rows with
    the same instrument column twice (same-lane repeated atomics, equal keys in the column-ordered copy, MATCH peers
    inside one lane).  Every path: default, two-product, attitude atomics, instrument copy, and a Zipf case (MATCH)."""
    gsr = gsr_mod()

    def scramble(cfg, d):
        rng = np.random.default_rng(77)
        rp = synth.star_rowptr(cfg).numpy()
        perm = np.concatenate([rp[s] + rng.permutation(rp[s + 1] - rp[s]) for s in range(cfg.n_stars)])
        out = dict(d)
        for k in ("values", "matrixIndexAstro", "matrixIndexAtt", "instrCol", "noise"):
            out[k] = np.ascontiguousarray(d[k][perm])
        assert np.array_equal(out["matrixIndexAstro"], d["matrixIndexAstro"])       # still sorted by star
        assert (np.diff(out["matrixIndexAtt"]) < 0).mean() > 0.3                      # no longer by time
        rows = rng.choice(len(perm), len(perm) // 20, replace=False)
        out["instrCol"][rows, 4] = out["instrCol"][rows, 1]
        return out

    plain = synth.SynthConfig("shuf", 3_000, 4_000, 300, obs_per_star=90, seed=51)
    zipf = synth.SynthConfig("shuf_zipf", 6_000, 3_000, 60_000, obs_powerlaw=(2.0, 10, 2000), att_bursts=(200, 2e-3, 0.7),
                             instr_zipf=1.1, seed=52)      # the shape of test_skewed_shape_match_red_and_table
    for cfg, flag_list in ((plain, (0, gsr.GSR_FLAG_NO_FUSE, gsr.GSR_FLAG_NO_ATT_COPY, gsr.GSR_FLAG_INS_COPY)),
                           (zipf, (0, gsr.GSR_FLAG_NO_FUSE))):
        d = scramble(cfg, np_inputs(cfg))
        S, _ = oracle_system(cfg, d)
        b = make_b(S, d)
        for flags in flag_list:
            with make_gpu(S, d, b, flags=flags) as G:
                info = G.gsr_path_info()
                assert bool(info & gsr.GSR_PATH_INSTR_MATCH) == (cfg is zipf)
                assert bool(info & gsr.GSR_PATH_INS_COPY) == (flags == gsr.GSR_FLAG_INS_COPY)
                check_aprods(S, G, seed=flags)
        S.precondition()
        ro = S.lsqr(b, 25, 0.0, 0.0)
        for flags in flag_list:
            with make_gpu(S, {**d, "values": S.V}, b, flags=flags) as G:      # the preconditioned matrix
                r = G.gsr_lsqr(25, 0.0, 0.0)
                assert (r.istop, r.itn) == (ro.istop, ro.itn) == (7, 25)
                assert rel(r.x.cpu().numpy() * S.p, ro.x) <= X_TOL, (cfg.name, flags)


def test_large_full_size_every_element():
    """BASELINE configs[4] at full size (500 M rows + 10,000 constraint rows x 1,000 non-zeros, ~170 GB resident) in the
    launch configuration bench.py times: every output of aprod1 (observation and constraint rows) and every output of
    aprod2 against the chunk-streamed oracle ("oracle parity on aprod only, chunk-streamed")."""
    import bench
    gsr = gsr_mod()
    torch.cuda.empty_cache()
    free, _ = torch.cuda.mem_get_info()
    if free < 183e9:
        pytest.skip("needs a whole 180 GB B200")
    cfg = synth.large()
    dv = torch.device("cuda", 0)
    m = int(synth.star_rowptr(cfg)[-1])
    with gsr.Gsr(m, cfg.n_stars, cfg.n_dof_att, cfg.n_instr, cfg.n_con, cfg.n_con * cfg.con_nnz) as G:
        bench.build_on_device(cfg, G, dv, torch, synth)
        assert G.gsr_path_info() & gsr.GSR_PATH_IC16
        g = torch.Generator(device="cuda").manual_seed(6)
        x = torch.randn(G.n, dtype=torch.float64, device=dv, generator=g)
        y = torch.randn(G.m_tot, dtype=torch.float64, device=dv, generator=g)
        y1 = G.gsr_aprod1(x, torch.zeros(G.m_tot, dtype=torch.float64, device=dv))
        x2 = G.gsr_aprod2(y, torch.zeros(G.n, dtype=torch.float64, device=dv))
        # constraint rows alone through the oracle (an oracle system without observation rows)
        rp, cc, cv = (t.cpu().numpy() for t in synth.constraints(cfg, dv))
        e = np.zeros((0, 24))
        Sc = oracle.OracleSystem(cfg.n_stars, cfg.n_dof_att, cfg.n_instr, e, np.zeros(0, np.int64), np.zeros(0, np.int64),
                                 np.zeros((0, 6), np.int32), rp, cc, cv)
        xc = x.cpu().numpy()
        yc, abc = Sc.aprod1(xc, np.zeros(cfg.n_con), want_abs=True)
        assert np.all(np.abs(y1[m:].cpu().numpy() - yc) <= APROD_TOL * abc)
        x2c, ab2c = Sc.aprod2(y[m:].cpu().numpy(), np.zeros(G.n), want_abs=True)
        # observation rows, chunk by chunk; the constraint rows' share of A^T y and of its bound is added to the reference
        worst1, err2 = stream_oracle_aprods(cfg, G, x, y[:m], y1[:m], x2, chunk_stars=10_000, x_extra=x2c, ab_extra=ab2c)
        assert float(err2.max()) <= APROD_TOL, float(err2.max())
        print(f"large every element: aprod1 worst {worst1:.2e}, aprod2 worst {float(err2.max()):.2e} (x 1e-12 bound)")


def test_skewed_full_size_every_element():
    """BASELINE configs[3] at full size (literal alpha = 2: 53 M rows, power-law rows per star, bursty attitude starts, 60,000
    Zipf columns: the MATCH variant, global REDs and the shared-memory table together): every output of both products
    against the chunk-streamed oracle."""
    import bench
    gsr = gsr_mod()
    cfg = synth.skewed()
    dv = torch.device("cuda", 0)
    m = int(synth.star_rowptr(cfg)[-1])
    with gsr.Gsr(m, cfg.n_stars, cfg.n_dof_att, cfg.n_instr) as G:
        bench.build_on_device(cfg, G, dv, torch, synth)
        assert G.gsr_path_info() & gsr.GSR_PATH_INSTR_MATCH
        g = torch.Generator(device="cuda").manual_seed(7)
        x = torch.randn(G.n, dtype=torch.float64, device=dv, generator=g)
        y = torch.randn(m, dtype=torch.float64, device=dv, generator=g)
        y1 = G.gsr_aprod1(x, torch.zeros(m, dtype=torch.float64, device=dv))
        x2 = G.gsr_aprod2(y, torch.zeros(G.n, dtype=torch.float64, device=dv))
        worst1, err2 = stream_oracle_aprods(cfg, G, x, y, y1, x2, chunk_stars=20_000)
        assert float(err2.max()) <= APROD_TOL, float(err2.max())
        print(f"skewed every element: aprod1 worst {worst1:.2e}, aprod2 worst {float(err2.max()):.2e} (x 1e-12 bound)")


@pytest.mark.parametrize("n_instr", [65_536, 65_537])
def test_instrument_column_width_boundary(n_instr):
    """65,536 columns still fit 2 bytes (the last column is 65,535), 65,537 do not: 4-byte columns, and the opt-in
    column-ordered copy is silently not built.  Both with and without GSR_FLAG_INS_COPY."""
    gsr = gsr_mod()
    cfg = synth.SynthConfig("edge", 600, 500, n_instr, obs_per_star=30, seed=41)
    S, d = oracle_system(cfg)
    for i in (5, 777, 17_999):                   # make sure the last column is in use (the rows keep 6 distinct columns)
        assert n_instr - 1 not in d["instrCol"][i]
        d["instrCol"][i, 3] = n_instr - 1
    S, _ = oracle_system(cfg, d)
    b = make_b(S, d)
    for flags in (0, gsr.GSR_FLAG_INS_COPY):
        with make_gpu(S, d, b, flags=flags) as G:
            info = G.gsr_path_info()
            assert bool(info & gsr.GSR_PATH_IC16) == (n_instr <= 65_536)
            assert bool(info & gsr.GSR_PATH_INS_COPY) == (flags != 0 and n_instr <= 65_536)
            check_aprods(S, G, seed=8)
            G.gsr_precondition()
    S.precondition()
    with make_gpu(S, {**d, "values": S.V}, b, flags=gsr.GSR_FLAG_INS_COPY) as G:   # the preconditioned matrix through LSQR
        r = G.gsr_lsqr(15, 0.0, 0.0)
        ro = S.lsqr(b, 15, 0.0, 0.0)
        assert rel(r.x.cpu().numpy() * S.p, ro.x) <= X_TOL


def test_small_config_lsqr():
    """BASELINE configs[1] (20 M rows; SURVEY 8(d) asks for full parity on Small): gsr_lsqr against the oracle's LSQR on
    the same bytes.  The preconditioned system reaches the rounding floor near iteration 40 (1 + test2 <= 1, istop 5),
    so (reading R19) x / se / trace parity is taken at a fixed 25 iterations, before the floor, and the run
    "to convergence or 2,000 iterations" of the config must stop with the same istop within +-2 iterations.  The two
    oracle solves run side by side on two host threads."""
    from concurrent.futures import ThreadPoolExecutor
    gsr = gsr_mod()
    cfg = synth.small()
    dv = torch.device("cuda", 0)
    d = {k: v.cpu().numpy() for k, v in synth.generate(cfg, dv).items()}      # generated on the device, same bytes both sides
    S = oracle.OracleSystem(cfg.n_stars, cfg.n_dof_att, cfg.n_instr, d["values"], d["matrixIndexAstro"],
                            d["matrixIndexAtt"], d["instrCol"])
    b = S.aprod1(d["x_true"], d["noise"])
    with gsr.Gsr(S.m, cfg.n_stars, cfg.n_dof_att, cfg.n_instr) as G:
        G.gsr_upload(d["values"], d["matrixIndexAstro"], d["matrixIndexAtt"], d["instrCol"], b)
        G.gsr_precondition()
        S.precondition()
        np.testing.assert_allclose(G.gsr_get_colscale().cpu().numpy(), S.p, rtol=P_TOL, atol=0)
        with ThreadPoolExecutor(2) as pool:
            f25 = pool.submit(S.lsqr, b, 25, 0.0, 0.0, 0.0, True)
            fconv = pool.submit(S.lsqr, b, 2000, 0.0, 0.0)
            r = G.gsr_lsqr(25, 0.0, 0.0)
            tr = G.gsr_get_trace()
            rc = G.gsr_lsqr(2000, 0.0, 0.0)
            ro, roc = f25.result(), fconv.result()
        assert (r.istop, r.itn) == (ro.istop, ro.itn) == (7, 25)
        assert rel(r.x.cpu().numpy(), ro.x) <= X_TOL
        assert rel(r.se.cpu().numpy(), ro.se) <= SE_TOL
        np.testing.assert_allclose(tr[:, 0], ro.trace[:, 0], rtol=1e-9)      # rnorm
        np.testing.assert_allclose(tr[:, 2], ro.trace[:, 2], rtol=1e-9)      # anorm
        np.testing.assert_allclose(tr[:, 4], ro.trace[:, 4], rtol=1e-9)      # xnorm
        assert rc.istop == roc.istop and rc.istop != 7, (rc.istop, roc.istop)
        assert abs(rc.itn - roc.itn) <= 2, (rc.itn, roc.itn)
        # The paper's own form of validation (section 6): mean +- std of the differences of the solution and of its
        # standard errors per section between two codes (Table 1), and the ratio
        # q = |dx| / sqrt(se_1^2 + se_2^2) < 1 for every unknown (Eq. 5) -- here CUDA path vs oracle.
        xg, sg = rc.x.cpu().numpy(), rc.se.cpu().numpy()
        na, nd = 5 * cfg.n_stars, 3 * cfg.n_dof_att
        for name, sl in (("astro", slice(0, na)), ("att", slice(na, na + nd)), ("instr", slice(na + nd, S.n - 1)),
                         ("glob", slice(S.n - 1, S.n))):
            dx, ds = xg[sl] - roc.x[sl], sg[sl] - roc.se[sl]
            q = np.abs(dx) / np.sqrt(sg[sl] ** 2 + roc.se[sl] ** 2)
            print(f"paper-style check, {name}: dx {dx.mean():.2e} +- {dx.std():.2e}, dse {ds.mean():.2e} +- {ds.std():.2e}, "
                  f"max q {q.max():.2e}")
            assert q.max() < 1.0, name
        assert rel(rc.x.cpu().numpy(), roc.x) <= X_TOL_CONVERGED
        assert rel(rc.x.cpu().numpy(), d["x_true"]) <= 1e-3


def test_skewed_shape_match_red_and_table():
    """Skewed-shaped (BASELINE configs[3]): power-law rows per star, bursty attitude times and 60,000 Zipf(1.1)
    instrument columns, so the variant that pre-sums equal columns inside a warp (MATCH) runs with BOTH the
    shared-memory table (the head of the Zipf distribution) and global REDs (its tail), in the fused and in the
    two-product form; run-to-run spread of x under the atomics is reported against the tolerance."""
    gsr = gsr_mod()
    # well posed on purpose (x parity at 1e-9 presumes it): every attitude coefficient is observed
    cfg = synth.SynthConfig("skew_s", 6_000, 3_000, 60_000, obs_powerlaw=(2.0, 10, 2000), att_bursts=(200, 2e-3, 0.7),
                            instr_zipf=1.1, seed=21)
    S, d = oracle_system(cfg)
    assert d["instrCol"].max() > 16_384             # columns beyond every shared-memory table in use
    b = make_b(S, d)
    for flags in (gsr.GSR_FLAG_NO_FUSE, 0):
        with make_gpu(S, d, b, flags=flags) as G:
            assert G.gsr_path_info() & gsr.GSR_PATH_INSTR_MATCH
            check_aprods(S, G)
            if flags == 0:
                G.gsr_precondition()
                S.precondition()
                ro = S.lsqr(b, 30, 0.0, 0.0)
                xs = []
                for _ in range(3):
                    r = G.gsr_lsqr(30, 0.0, 0.0)
                    assert (r.istop, r.itn) == (ro.istop, ro.itn) == (7, 30)
                    xs.append(r.x.cpu().numpy())
                    assert rel(xs[-1], ro.x) <= X_TOL
                spread = max(np.max(np.abs(xs[0] - xk)) for xk in xs[1:])
                assert spread <= X_TOL * np.linalg.norm(ro.x)
    # the preconditioned matrix (flags = 0 above scaled S) in the two-product form as well
    with make_gpu(S, {**d, "values": S.V}, b, flags=gsr.GSR_FLAG_NO_FUSE) as G:
        r = G.gsr_lsqr(30, 0.0, 0.0)
        ro2 = S.lsqr(b, 30, 0.0, 0.0)
        assert rel(r.x.cpu().numpy() * S.p, ro2.x) <= X_TOL


def test_constraint_rows_at_size():
    """Constraint kernels beyond one warp pass and one grid pass: 2,500 rows x 160 non-zeros on a
    small system (both loops of k_con_aprod1/2 iterate; LSQR through the fused and the two-product form), then the
    Large config's own tail -- 10,000 rows x 1,000 random astro columns of 2.5 M stars -- against the oracle on the
    constraint rows alone (observation rows only for the first stars)."""
    gsr = gsr_mod()
    cfg = synth.SynthConfig("con_mid", 1_500, 600, 40, obs_per_star=30, n_con=2_500, con_nnz=160, seed=31)
    S, d = oracle_system(cfg)
    b = make_b(S, d)
    for flags in (0, gsr.GSR_FLAG_NO_FUSE):
        with make_gpu(S, d, b, flags=flags) as G:
            check_aprods(S, G)
    with make_gpu(S, d, b) as G:
        G.gsr_precondition()
        S.precondition()
        check_aprods_scaled(S, G)
        r = G.gsr_lsqr(25, 0.0, 0.0)
        ro = S.lsqr(b, 25, 0.0, 0.0)
        assert (r.istop, r.itn) == (ro.istop, ro.itn) == (7, 25)
        assert rel(r.x.cpu().numpy(), ro.x) <= X_TOL
    # Large's tail: columns drawn over 5 * 2,500,000 astro unknowns
    big = synth.large()
    cfgL = synth.SynthConfig("large_tail", big.n_stars, 2_000, 600, obs_per_star=40, n_con=big.n_con, con_nnz=big.con_nnz,
                             seed=big.seed)
    rp, cc, cv = (t.numpy() for t in synth.constraints(cfgL))
    sub = synth.generate_rows(cfgL, 0, 500)          # rows for the first 500 stars only; the others have none
    P = {k: sub[k].numpy() for k in ("values", "matrixIndexAstro", "matrixIndexAtt", "instrCol")}
    SL = oracle.OracleSystem(cfgL.n_stars, cfgL.n_dof_att, cfgL.n_instr, P["values"], P["matrixIndexAstro"],
                             P["matrixIndexAtt"], P["instrCol"], rp, cc, cv)
    assert SL.n_con == 10_000 and len(cc) == 10_000_000
    with make_gpu(SL, P, np.zeros(SL.m_tot)) as G:
        rng = np.random.default_rng(2)
        x, y = rng.standard_normal(SL.n), rng.standard_normal(SL.m_tot)
        y1 = G.gsr_aprod1(dev(x), dev(y)).cpu().numpy()
        y1o, ab = SL.aprod1(x, y, want_abs=True)
        assert np.all(np.abs(y1 - y1o) <= APROD_TOL * ab)
        x2 = G.gsr_aprod2(dev(y), dev(x)).cpu().numpy()
        x2o, ab2 = SL.aprod2(y, x, want_abs=True)
        assert np.all(np.abs(x2 - x2o) <= APROD_TOL * ab2)


def test_reupload_with_constraints_is_clean():
    """upload, precondition, upload again, precondition: the constraint rows must come again with every upload (the
    first gsr_precondition scaled them in place) and the second solve equals the first."""
    gsr = gsr_mod()
    cfg = CASES["mini_con"]["cfg"]
    S, d = oracle_system(cfg)
    b = make_b(S, d)
    with make_gpu(S, d, b) as G:
        G.gsr_precondition()
        p1 = G.gsr_get_colscale().cpu().numpy()
        x1 = G.gsr_lsqr(20, 0.0, 0.0).x.cpu().numpy()
        G.gsr_upload(np.ascontiguousarray(d["values"]), np.ascontiguousarray(d["matrixIndexAstro"]),
                     np.ascontiguousarray(d["matrixIndexAtt"]), np.ascontiguousarray(d["instrCol"]), b)
        with pytest.raises(gsr.GsrError) as e:           # constraints were discarded by the upload
            G.gsr_precondition()
        assert e.value.code == gsr.GSR_ESTATE
        G.gsr_upload_constraints(S.con_rowptr, S.con_col, S.con_val)
        G.gsr_precondition()
        np.testing.assert_allclose(G.gsr_get_colscale().cpu().numpy(), p1, rtol=1e-14, atol=0)   # att / instr sums use atomics
        x2 = G.gsr_lsqr(20, 0.0, 0.0).x.cpu().numpy()
        assert rel(x2, x1) <= 1e-11
        S.precondition()
        assert rel(x2, S.lsqr(b, 20, 0.0, 0.0).x) <= X_TOL


@pytest.mark.parametrize("flag", ["NO_ATT_COPY", "NO_FUSE", "NO_TEX", "INS_COPY", "INS_COPY+NO_FUSE"])
@pytest.mark.parametrize("case", ["mini_con", "zipf_hot", "ragged_tail"])
def test_fallback_paths(flag, case):
    """gsr_layout.flags, per handle and in-process: the low-memory path (no block-time-ordered attitude copy:
    attitude REDs inside k_aprod2, two-product iteration), the two-product form of the iteration on the default
    layout, and the fused pass without texture objects (the path systems with n >= 2^27 take) all give the
    oracle's results."""
    gsr = gsr_mod()
    fl = {"NO_ATT_COPY": gsr.GSR_FLAG_NO_ATT_COPY, "NO_FUSE": gsr.GSR_FLAG_NO_FUSE, "NO_TEX": gsr.GSR_FLAG_NO_TEX,
          "INS_COPY": gsr.GSR_FLAG_INS_COPY, "INS_COPY+NO_FUSE": gsr.GSR_FLAG_INS_COPY | gsr.GSR_FLAG_NO_FUSE}[flag]
    cfg = CASES[case]["cfg"]
    S, d = oracle_system(cfg)
    b = make_b(S, d)
    with make_gpu(S, d, b, flags=fl) as G:
        info = G.gsr_path_info()
        assert bool(info & gsr.GSR_PATH_ATT_COPY) == (flag != "NO_ATT_COPY")
        assert bool(info & gsr.GSR_PATH_FUSED) == (flag in ("NO_TEX", "INS_COPY"))
        assert bool(info & gsr.GSR_PATH_TEX) == (flag != "NO_TEX")
        assert bool(info & gsr.GSR_PATH_INSTR_MATCH) == (case == "zipf_hot")
        # the column-ordered instrument copy is opt-in and needs unskewed columns
        assert bool(info & gsr.GSR_PATH_INS_COPY) == (flag.startswith("INS_COPY") and case != "zipf_hot")
        check_aprods(S, G)
        G.gsr_precondition()
        S.precondition()
        r = G.gsr_lsqr(25, 0.0, 0.0)
        ro = S.lsqr(b, 25, 0.0, 0.0)
        assert r.itn == ro.itn == 25 and r.istop == ro.istop == 7
        assert rel(r.x.cpu().numpy(), ro.x) <= X_TOL
        assert rel(r.se.cpu().numpy(), ro.se) <= SE_TOL
        # kernels that exist only on the default path
        if flag == "NO_ATT_COPY":
            with pytest.raises(gsr.GsrError):
                G.gsr_time_aprod(gsr.GSR_TIME_K_APROD2_ATT, 1)
        if flag not in ("NO_TEX", "INS_COPY"):
            with pytest.raises(gsr.GsrError):
                G.gsr_time_aprod(gsr.GSR_TIME_K_FUSED, 1)
        if not (info & gsr.GSR_PATH_INS_COPY):
            with pytest.raises(gsr.GsrError):
                G.gsr_time_aprod(gsr.GSR_TIME_K_INS_SCATTER, 1)


# ----------------------------------------------------------------------------- model variants
VARIANT_LAYOUTS = [   # (n_astro_par, n_att_par, n_instr_par, n_glob)
    (0, 12, 6, 0),    # attitude + instrumental only (the paper's 40 / 300 GB datasets)
    (5, 0, 0, 0),     # astrometric only (100 GB dataset)
    (5, 12, 6, 0),    # no global part (350 GB dataset; "so far ... we have run without computing a global part")
    (5, 12, 6, 5),    # five global parameters
    (3, 12, 4, 2),
    (2, 0, 1, 16),    # widest global section the library takes
]


def variant_cfg(widths, shape):
    na, nt, ni, ng = widths
    base = {"ragged": synth.mini(seed=21, n_stars=37, obs=23, n_dof_att=64, n_instr=10),                 # 851 rows
            "powerlaw": synth.SynthConfig("plv", 400, 300, 50, obs_powerlaw=(2.0, 8, 200), att_bursts=(5, 1e-2, 0.9),
                                          instr_zipf=1.1, seed=22),                                       # stars cut by tile edges
            "multi_cta": synth.SynthConfig("mc", 3_000, 2_000, 70_000, obs_per_star=41, seed=23)}[shape]  # 123,000 rows, 4-byte columns
    return dataclasses.replace(base, n_astro_par=na, n_att_par=nt, n_instr_par=ni, n_glob=ng)


@pytest.mark.parametrize("shape", ["ragged", "powerlaw", "multi_cta"])
@pytest.mark.parametrize("widths", VARIANT_LAYOUTS)
def test_model_variants_aprod_and_precondition(widths, shape):
    """Layouts other than 5/12/6/1 (general kernels k_aprod1_gen / k_aprod2_gen): sizes, star row pointer, both products
    element by element, the preconditioner and the scaled coefficients against the oracle."""
    cfg = variant_cfg(widths, shape)
    S, d = oracle_system(cfg)
    b = make_b(S, d)
    with make_gpu(S, d, b) as G:
        assert G.n == S.n == cfg.n and G.m_tot == S.m_tot
        info = G.gsr_path_info()
        # 5/12/6/N_Glob and 0/12/6/0 (the section subsets of the paper's datasets, any number of global columns) share the
        # specialised kernels and the fused iteration with the production layout; the other layouts run the general kernels
        assert bool(info & gsr_mod().GSR_PATH_FUSED) == (widths[:3] == (5, 12, 6) or widths == (0, 12, 6, 0))
        assert bool(info & gsr_mod().GSR_PATH_ATT_COPY) == (widths[1] == 12)   # the attitude kernel serves every layout
        if widths[0]:
            rp = G.gsr_get_star_rowptr().cpu().numpy()
            assert np.array_equal(rp, d["rowptr"])
        else:
            with pytest.raises(gsr_mod().GsrError):
                G.gsr_get_star_rowptr()
        check_aprods(S, G, seed=3)
        G.gsr_precondition()
        po = S.precondition()
        np.testing.assert_allclose(G.gsr_get_colscale().cpu().numpy(), po, rtol=P_TOL, atol=0)
        V, _ = G.gsr_get_values()
        assert V.shape == S.V.shape
        np.testing.assert_allclose(V.cpu().numpy(), S.V, rtol=P_TOL, atol=0)
        check_aprods_scaled(S, G)


@pytest.mark.parametrize("widths", VARIANT_LAYOUTS)
def test_model_variants_lsqr(widths):
    cfg = variant_cfg(widths, "ragged")
    S, d, G, r, ro = lsqr_both(cfg, 25, 0.0, 0.0)
    with G:
        assert (r.istop, r.itn) == (ro.istop, ro.itn) == (7, 25)
        assert rel(r.x.cpu().numpy(), ro.x) <= X_TOL
        assert rel(r.se.cpu().numpy(), ro.se) <= SE_TOL
        for a, bb in ((r.rnorm, ro.rnorm), (r.anorm, ro.anorm), (r.acond, ro.acond), (r.xnorm, ro.xnorm)):
            assert abs(a - bb) <= 1e-9 * abs(bb)
    # to convergence: same stop code, itn within 2
    S, d, G, r, ro = lsqr_both(cfg, 400, 1e-12, 1e-12)
    with G:
        assert r.istop == ro.istop and abs(r.itn - ro.itn) <= 2, (r.istop, r.itn, ro.istop, ro.itn)
        assert rel(r.x.cpu().numpy(), ro.x) <= X_TOL_CONVERGED


@pytest.mark.parametrize("flag", ["NO_FUSE", "NO_TEX"])
@pytest.mark.parametrize("widths", [(5, 12, 6, 0), (0, 12, 6, 0), (5, 12, 6, 5), (5, 12, 6, 16)])
def test_fast_variant_layouts_fallback_paths(widths, flag):
    """The two non-production layouts that run the specialised kernels, in the two-product form and without textures."""
    gsr = gsr_mod()
    cfg = variant_cfg(widths, "multi_cta")
    S, d = oracle_system(cfg)
    b = make_b(S, d)
    with make_gpu(S, d, b, flags={"NO_FUSE": gsr.GSR_FLAG_NO_FUSE, "NO_TEX": gsr.GSR_FLAG_NO_TEX}[flag]) as G:
        assert bool(G.gsr_path_info() & gsr.GSR_PATH_FUSED) == (flag == "NO_TEX")
        check_aprods(S, G, seed=6)
        G.gsr_precondition()
        S.precondition()
        r = G.gsr_lsqr(15, 0.0, 0.0)
        ro = S.lsqr(b, 15, 0.0, 0.0)
        assert (r.istop, r.itn) == (ro.istop, ro.itn) == (7, 15)
        assert rel(r.x.cpu().numpy(), ro.x) <= X_TOL
        assert rel(r.se.cpu().numpy(), ro.se) <= SE_TOL


@pytest.mark.parametrize("widths", [(0, 12, 6, 0), (3, 12, 4, 2)])
def test_model_variants_without_attitude_copy(widths):
    """GSR_FLAG_NO_ATT_COPY on a non-production layout: the attitude section goes through the REDs of k_aprod2_gen."""
    gsr = gsr_mod()
    Sp, dp = oracle_system(variant_cfg(widths, "powerlaw"))      # stars cut by tile edges, bursts: products only (the
    with make_gpu(Sp, dp, make_b(Sp, dp), flags=gsr.GSR_FLAG_NO_ATT_COPY) as G:   # Zipf / burst system is too ill-posed
        check_aprods(Sp, G, seed=5)                              # for the 1e-9 bound on x)
    cfg = variant_cfg(widths, "ragged")
    S, d = oracle_system(cfg)
    b = make_b(S, d)
    with make_gpu(S, d, b, flags=gsr.GSR_FLAG_NO_ATT_COPY) as G:
        assert not (G.gsr_path_info() & gsr.GSR_PATH_ATT_COPY)
        check_aprods(S, G, seed=4)
        G.gsr_precondition()
        S.precondition()
        r = G.gsr_lsqr(25, 0.0, 0.0)
        ro = S.lsqr(b, 25, 0.0, 0.0)
        assert (r.istop, r.itn) == (ro.istop, ro.itn) == (7, 25)
        assert rel(r.x.cpu().numpy(), ro.x) <= X_TOL


def test_model_variants_global_columns_bit_reproducible():
    """Every global column is reduced in a fixed order (warp -> CTA -> one block), as gamma is in production: in the
    general kernels (3/12/4/5) and in the specialised ones (5/12/6/5)."""
    for widths in ((3, 12, 4, 5), (5, 12, 6, 5)):
        cfg = variant_cfg(widths, "multi_cta")
        S, d = oracle_system(cfg)
        b = make_b(S, d)
        with make_gpu(S, d, b) as G:
            y = torch.from_numpy(np.random.default_rng(0).standard_normal(S.m_tot)).cuda()
            outs = [G.gsr_aprod2(y, torch.zeros(S.n, dtype=torch.float64, device="cuda")).cpu().numpy() for _ in range(3)]
            na = widths[0] * cfg.n_stars
            for o in outs[1:]:
                assert np.array_equal(o[:na], outs[0][:na])
                assert np.array_equal(o[-5:], outs[0][-5:])


def test_layout_width_validation():
    gsr = gsr_mod()
    for bad in ((6, 12, 6, 1), (5, 8, 6, 1), (5, 12, 7, 1), (5, 12, 6, 17), (0, 0, 0, 0), (-1, 12, 6, 1)):
        with pytest.raises(gsr.GsrError) as e:
            gsr.Gsr(10, 2, 8, 8, n_astro_par=bad[0], n_att_par=bad[1], n_instr_par=bad[2], n_glob=bad[3])
        assert e.value.code == gsr.GSR_EINVAL
