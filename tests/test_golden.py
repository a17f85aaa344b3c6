"""Oracle vs the paper's printed fp64 agreement bounds (Table 1; tests/golden/paper_table1.txt).
Two independent fp64 formulations inside oracle/ must agree about as closely as BARD and Pinocchio do."""
import os

import numpy as np
import pytest

import oracle
from paper_2605_31481_b200 import workloads as W

HERE = os.path.dirname(os.path.abspath(__file__))
COL = {0: 0, 2: 1, 1: 2, 3: 3}          # config -> column of the fixture
SLACK = 50.0                             # different robots, different link sizes: a small multiple of the bound


def table1():
    out = {}
    for line in open(os.path.join(HERE, "golden", "paper_table1.txt")):
        if line.startswith("#") or not line.strip():
            continue
        p = line.split()
        out[p[0]] = [float(x) for x in p[1:]]
    return out


@pytest.mark.parametrize("cfg", [0, 1, 2, 3])
def test_two_formulations_agree_within_table1(cfg):
    T = table1()
    desc = W.config_robot(cfg)
    o = oracle.Oracle(desc)
    q, qd, qdd = (a.astype(np.float64) for a in W.config_states(cfg, 1000))
    c = COL[cfg]
    # FK: explicit 4x4 products vs Rodrigues constants eq. (2)-(5)
    assert np.max(np.abs(o.fk(q) - o.fk_rodrigues(q))) <= SLACK * T["FK"][c]
    # CRBA vs column k = RNEA(q, 0, e_k; g = 0)
    M = o.crba(q)
    g0 = oracle.Oracle(_zero_g(desc))
    nv = desc.nv
    cols = np.stack([g0.rnea(q, np.zeros_like(qd), np.tile(np.eye(nv)[:, k:k + 1], (1, q.shape[1]))) for k in range(nv)], 1)
    scale = max(1.0, float(np.max(np.abs(M))))
    assert np.max(np.abs(M - cols)) <= SLACK * T["CRBA"][c] * scale
    # RNEA(q, qd, qdd) - RNEA(q, qd, 0) = M qdd
    d = o.rnea(q, qd, qdd) - o.rnea(q, qd, np.zeros_like(qdd))
    Mq = np.einsum("ijb,jb->ib", M, qdd)
    assert np.max(np.abs(d - Mq)) <= SLACK * T["RNEA"][c] * max(1.0, float(np.max(np.abs(Mq))))


def _zero_g(desc):
    import copy
    d = copy.copy(desc)
    d.gravity = np.zeros(3)
    return d
