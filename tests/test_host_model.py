"""CPU tests of the C-ABI library's host logic: it loads, exports every symbol include/bard.h declares,
validates descriptions, and its level schedule / index tables are BIT-EXACT against the oracle's
(which derives them by a different route).  No kernel is launched here."""
import ctypes as C
import os
import re

import numpy as np
import pytest

import oracle
from paper_2605_31481_b200 import binding, workloads as W

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
INT_TABLES = ["LEVEL_PTR", "LEVEL_BODY", "BODY_LEVEL", "PARENT_SLOT", "Q_OFF", "V_OFF", "DOF_BODY", "ANC_MASK"]


def test_library_exports_every_declared_symbol():
    hdr = open(os.path.join(ROOT, "include", "bard.h")).read()
    declared = set(re.findall(r"\b(bard_[a-z0-9_]+)\s*\(", hdr))
    assert declared == set(binding.EXPORTS)
    L = binding.lib()
    for name in declared:
        assert hasattr(L, name), name


def _robots():
    out = [W.config_robot(c) for c in range(4)]
    for seed in range(12):
        shape = ["random", "chain", "star", "unbalanced"][seed % 4]
        out.append(W.random_tree(100 + seed, nb=3 + 5 * seed, shape=shape, free_root=(seed % 3 == 0)))
    out.append(W.random_tree(999, nb=64, shape="random"))
    return out


@pytest.mark.parametrize("idx", range(17))
def test_tables_bit_exact_vs_oracle(idx):
    desc = _robots()[idx]
    m = binding.Model(desc, device=-1)
    o = oracle.Oracle(desc)
    assert (m.nb, m.nq, m.nv, m.nlevels) == (o.nb, o.nq, o.nv, o.nlevels)
    for name in INT_TABLES:
        a, b = m.table(name), o.table(name)
        assert a.shape == b.shape, name
        assert np.array_equal(a.astype(np.uint64), b.astype(np.uint64)), name


@pytest.mark.parametrize("idx", [0, 3, 5, 9])
def test_rodrigues_constants_vs_oracle(idx):
    desc = _robots()[idx]
    m = binding.Model(desc, device=-1)
    ref = oracle.Oracle(desc).rodrigues().reshape(-1)
    got = m.table("RODRIGUES").astype(np.float64)
    assert np.max(np.abs(got - ref)) <= 1e-6


def test_config_level_widths():
    # widths per level of the four configs
    want = {0: [1] * 7, 1: [1, 4, 4, 4], 2: [1, 1, 3, 3, 2, 2], 3: [1, 3, 3, 5, 4, 4, 4]}
    for cfg, w in want.items():
        m = binding.Model(W.config_robot(cfg), device=-1)
        assert np.diff(m.table("LEVEL_PTR")).tolist() == w


def test_validation_errors():
    d = W.config_robot(0)
    bad = W.config_robot(0)
    bad.parent = np.array([-1, 0, 1, 5, 3, 4, 5], np.int32)
    with pytest.raises(binding.BardError) as ei:
        binding.Model(bad, device=-1)
    assert ei.value.code == 2
    bad = W.config_robot(0)
    bad.joint_type = np.array([0, 0, 9, 0, 0, 0, 0], np.int32)
    with pytest.raises(binding.BardError) as ei:
        binding.Model(bad, device=-1)
    assert ei.value.code == 1
    bad = W.config_robot(0)
    bad.mass = bad.mass.copy()
    bad.mass[2] = -1.0
    with pytest.raises(binding.BardError):
        binding.Model(bad, device=-1)
    bad.mass[2] = float("nan")
    with pytest.raises(binding.BardError):
        binding.Model(bad, device=-1)
    bad.mass[2] = 0.0                                # a massless link is legal (URDF frames behind fixed joints)
    binding.Model(bad, device=-1).close()
    bad = W.config_robot(0)
    bad.axis = bad.axis.copy()
    bad.axis[1] = 0.0
    with pytest.raises(binding.BardError):
        binding.Model(bad, device=-1)
    big = W.random_tree(5, nb=65)
    with pytest.raises(binding.BardError) as ei:
        binding.Model(big, device=-1)
    assert ei.value.code == 3
    # host-only model refuses to run operators; bad frame rejected
    m = binding.Model(d, device=-1)
    with pytest.raises(binding.BardError):
        m.fk(4, 1, 1)
    with pytest.raises(binding.BardError):
        m.set_frames([7])
    assert binding.lib().bard_status_string(2) == b"BARD_ERR_TOPOLOGY"


def test_free_joint_requires_identity_T_post():
    d = W.random_tree(3, nb=4, free_root=True)
    d.T_post = d.T_post.copy()
    d.T_post[0, 3] = 0.1
    with pytest.raises(binding.BardError):
        binding.Model(d, device=-1)


def test_options_are_fields_of_the_model_and_null_handles_are_refused(monkeypatch):
    """Knobs live in the model: the environment gives the default ONCE at bard_model_create, set_option overrides it,
    another model is unaffected; unknown keys and NULL handles return BARD_ERR_INVALID_ARG (never a crash)."""
    monkeypatch.setenv("BARD_SPEC_MIN_B", "777")
    a = binding.Model(W.config_robot(0), device=-1)
    monkeypatch.delenv("BARD_SPEC_MIN_B")
    b = binding.Model(W.config_robot(0), device=-1)
    assert a.get_option("spec_min_b") == 777 and b.get_option("spec_min_b") == -1
    a.set_option("spec_min_b", 5)
    assert a.get_option("spec_min_b") == 5 and b.get_option("spec_min_b") == -1
    with pytest.raises(binding.BardError) as ei:
        a.set_option("no_such_knob", 1)
    assert ei.value.code == 1
    L = binding.lib()
    import ctypes as C
    v = C.c_int64()
    null = C.c_void_p()
    assert L.bard_model_set_option(null, b"pack", 1) == 1
    assert L.bard_model_get_option(null, b"pack", C.byref(v)) == 1
    # every operator entry point with a NULL model: an error code, not a segfault
    assert L.bard_fk(null, 4, None, None, None) == 1
    assert L.bard_jacobian(null, 4, None, None, None) == 1
    assert L.bard_rnea(null, 4, None, None, None, None, None) == 1
    assert L.bard_crba(null, 4, None, None, None) == 1
    assert L.bard_step(null, 4, None, None, None, None, None, None, None, None) == 1
    assert L.bard_euler_step(null, 4, 0.01, None, None, None, None) == 1
    assert L.bard_aba(null, 4, None, None, None, None, None, None) == 1
    assert L.bard_model_set_frames(null, 0, None, None) == 1
    assert L.bard_model_specialize(null, 1) == 1
