"""Shared test helpers: build oracle systems / dense expansions from synthetic inputs."""
import numpy as np

import oracle
from paper_2308_00778_b200 import synth


def np_inputs(cfg, device="cpu"):
    d = synth.generate(cfg, device)
    return {k: v.cpu().numpy() for k, v in d.items()}


def oracle_system(cfg, d=None):
    d = d or np_inputs(cfg)
    con = (d["con_rowptr"], d["con_col"], d["con_val"]) if cfg.n_con else (None, None, None)
    return oracle.OracleSystem(cfg.n_stars, cfg.n_dof_att, cfg.n_instr, d["values"],
                               d["matrixIndexAstro"], d["matrixIndexAtt"], d["instrCol"], *con, n_glob=cfg.n_glob,
                               n_astro_par=cfg.n_astro_par, n_att_par=cfg.n_att_par, n_instr_par=cfg.n_instr_par), d


def dense(S):
    """Dense expansion of the oracle's stored system through its column map."""
    A = np.zeros((S.m_tot, S.n))
    for i in range(S.m):
        for k in range(S.n_par):
            A[i, S.col(i, k)] += S.V[i, k]
    for r in range(S.n_con):
        for q in range(S.con_rowptr[r], S.con_rowptr[r + 1]):
            A[S.m + r, S.con_col[q]] += S.con_val[q]
    return A


def make_b(S, d):
    """b = A x_true + noise, formed by the oracle (inputs never come from the CUDA path)."""
    y0 = np.zeros(S.m_tot)
    y0[: S.m] = d["noise"]
    return S.aprod1(d["x_true"], y0)
