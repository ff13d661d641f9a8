"""Host-side checks of the C-ABI library (no GPU): it loads, exports every symbol include/fusefss.h declares,
compiles every spec to the shape the paper / the oracle fixes, and reports errors as codes."""
import ctypes as C
import os
import re

import numpy as np
import pytest

from workloads import specs

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def F():
    import __graft_entry__ as g
    g.build()
    import paper_2606_09551_b200 as F
    return F


def test_exports_every_declared_symbol(F):
    hdr = open(os.path.join(ROOT, "include", "fusefss.h")).read()
    declared = set(re.findall(r"\b(fusefss_[a-z0-9_]+)\s*\(", hdr))
    assert declared == set(F.SYMBOLS)
    raw = C.CDLL(F.LIB_PATH)
    for name in declared:
        assert hasattr(raw, name), name


ALL = [("relu16", lambda: specs.relu(16, 8)), ("gelu", specs.gelu), ("nexp", specs.nexp), ("recip", specs.recip),
       ("shift_relu", specs.shift_relu), ("rsqrt", specs.rsqrt), ("silu", specs.silu),
       ("toy", lambda: specs.toy(8, 3)), ("toy_masked", lambda: specs.toy(8, 3, True)),
       ("plain", specs.plain_default), ("single", specs.single_interval), ("nobits", specs.no_bits),
       ("full", specs.full_partition), ("shift_relu8", lambda: specs.shift_relu(8, 3)), ("ars", lambda: specs.ars(64, 12)),
       ("ars8", lambda: specs.ars(8, 3)), ("a2b8", lambda: specs.a2b_demo(8, 3)), ("a2b64", lambda: specs.a2b_demo(64, 12)),
       ("tiny1", lambda: specs.tiny_ring(1)), ("tiny2", lambda: specs.tiny_ring(2))]
ALL = ALL + [(nm + "_sp", (lambda mk=mk: specs.shared_prefix(mk()))) for nm, mk in ALL]      # variant 1 (DESIGN 9)
ALL = ALL + [(nm + "_xm", (lambda mk=mk: specs.input_masked_mul(mk()))) for nm, mk in ALL]  # variant bit 1 (DESIGN 10)
ALL = ALL + [(nm + "_xp", (lambda mk=mk: specs.public_point_horner(mk()))) for nm, mk in ALL[:40]]  # variant bit 2 (DESIGN 11)
ALL = ALL + [(nm + "_dense", (lambda mk=mk: specs.dense_table(mk()))) for nm, mk in ALL[:20] if nm in ("relu16", "toy", "toy_masked", "plain", "nobits", "full", "shift_relu8", "ars8")]  # variant bit 4 (DESIGN 14)
ALL = ALL + [(nm + "_et", (lambda mk=mk: specs.early_termination(mk()))) for nm, mk in ALL[:40] + ALL[-4:]]  # variant bit 3 (DESIGN 13)


# gate types AT the compiled limits (m = 63, p = 8, T = 64, 63 output bits; 32 AND gates = one message bit word in one round)
ALL = ALL + [("limits", specs.limits), ("limits_sp", lambda: specs.shared_prefix(specs.limits(n_pred=1))), ("limits_et", lambda: specs.early_termination(specs.limits())),
             ("limits_pw", specs.limits_piecewise), ("limits_pw_sp", lambda: specs.shared_prefix(specs.limits_piecewise()))]


@pytest.mark.parametrize("name,mk", ALL)
def test_compile_matches_oracle_shape(F, orc, name, mk):
    """Two independent compilers (DESIGN 4.3): same L_shape, atoms, key size, message sizes."""
    s = mk()
    P, O = F.Program(s), orc.Program(s)
    assert P.shape == O.shape
    for t in range(P.shape["T"]):
        assert P.atom(t) == O.atom(t)
    for count in (1, 31, 32, 33, 4096, 100003):
        assert P.key_bytes(count) == O.key_bytes(count)
        for q in range(P.post_rounds() + 1):
            assert P.post_msg_bytes(count, q) == O.post_msg_bytes(count, q)
    assert P.post_rounds() == O.post_rounds()
    assert P.online_bits() == O.online_bits()


@pytest.mark.parametrize("mk,kw", [(specs.limits, dict(m=64)), (specs.limits, dict(r=3, d=2)), (specs.limits, dict(n_pred=64)),
                                   (specs.limits_piecewise, dict(m=33)), (lambda: specs.shared_prefix(specs.limits()), {})])
def test_both_compilers_reject_beyond_the_limits(F, orc, mk, kw):
    """one step past each limit (m = 64 intervals, p = 9 payload words, T = 65 atoms, 33 AND gates in one round): FUSEFSS_E_SPEC from
    the library, NULL from the oracle's compiler -- never a truncated program; likewise the single-key construction of the T = 64 gate,
    whose predicates and boundaries together would need 125 points"""
    s = mk(**kw)
    with pytest.raises(Exception):
        F.Program(s)
    with pytest.raises(Exception):
        orc.Program(s)


def test_appendix_N_shape(F):
    """App. N: T = 2 atoms of width n, M = 3, p = 2, one Beaver multiplication."""
    P = F.Program(specs.relu(16, 8))
    assert (P.shape["T"], P.shape["M"], P.shape["p"], P.shape["M_A"], P.shape["M_B"], P.shape["G_mix"]) == (2, 3, 2, 1, 0, 0)
    assert P.shape["k"] == [16, 16]
    N = 1 << 16
    assert P.atom(0) == dict(k=16, c=0, is_theta=0, beta=0)
    assert P.atom(1) == dict(k=16, c=0, is_theta=1, beta=N // 2)


def test_key_bytes_formula(F):
    """DESIGN 4.4 / SURVEY 8(a): per element per party, unpadded: bitDCF(k) = 16(k+1) + 8, vecDCF(n,p) = 16 + n(16+8p) + 8p."""
    for mk in (specs.gelu, specs.silu, specs.shift_relu):
        s = mk()
        P = F.Program(s)
        sh = P.shape
        count = 1 << 20                                          # multiple of 32: no padding
        per = sum(16 * (k + 1) + 8 for k in sh["k"]) + 8 * sh["p"] + (sh["M"] - 1) * (16 + s.n * (16 + 8 * sh["p"]) + 8 * sh["p"])
        per += 8 + 8 * len(s.kappa_a) + (8 if sh["n_kb"] else 0) + 24 * sh["M_A"] + (24 if sh["M_B"] else 0) + (8 if sh["G_mix"] else 0) + 8 * sh["G_mix"]
        assert P.key_bytes(count) == per * count


def test_rejects_ill_formed_specs(F):
    good = specs.relu(16, 8)
    bad = specs.relu(16, 8)
    bad.alpha = [0]                                             # boundary must be > 0
    with pytest.raises(F.FuseFSSError):
        F.Program(bad)
    bad2 = specs.toy(8, 3)
    bad2.alpha = [5, 5, 9]                                      # not strictly increasing
    with pytest.raises(F.FuseFSSError):
        F.Program(bad2)
    bad3 = specs.relu(16, 8)
    bad3.n = 65
    with pytest.raises(F.FuseFSSError):
        F.Program(bad3)
    from test_oracle_gate import ill_formed_specs
    for why, s in ill_formed_specs():                           # the same list the oracle's compiler rejects
        with pytest.raises(F.FuseFSSError):
            F.Program(s)
            pytest.fail("accepted: " + why)
    with pytest.raises(F.FuseFSSError):
        F.Program(specs.dense_table(specs.gelu()))             # dense table: n <= 16 only
    assert F.Program(good).shape["T"] == 2
    assert F.lib.fusefss_key_bytes(None, 10) == 0
    assert F.lib.fusefss_strerror(-3) == b"party must be 0 or 1"


def test_argument_errors_without_gpu(F):
    P = F.Program(specs.relu(16, 8))
    # null pointers / bad party / zero count are rejected before any CUDA call
    assert F.lib.fusefss_eval_cmp(0, P._h, None, None, 10, None, None) == -1
    assert F.lib.fusefss_eval_cmp(2, P._h, 1, 1, 10, 1, None) == -3
    assert F.lib.fusefss_eval_lut(0, P._h, 1, 1, 0, 1, None) == -4
    assert F.lib.fusefss_keygen(P._h, None, None, 0, 0, 10, None, None, None) == -1
    Pn = F.Program(specs.no_bits())
    assert F.lib.fusefss_eval_cmp(0, Pn._h, 1, 1, 10, 1, None) == -7     # T = 0: call omitted
    Ps = F.Program(specs.single_interval())
    assert F.lib.fusefss_eval_lut(0, Ps._h, 1, 1, 10, 1, None) == -7     # m = 1: call omitted
    assert F.lib.fusefss_post(0, P._h, 1, 1, 1, 1, 10, 99, 1, 1, 1, 1, None) == -5
    assert F.lib.fusefss_gate_host(P._h, 1, 1, 1, 0, 10, 10, 1, 16, 1, 1, 1, 1, None) == -8    # workspace too small
    assert F.lib.fusefss_debug_set(b"no_such_knob", 1) == -9 and F.lib.fusefss_debug_set(b"force_g", 0) == 0
    assert F.lib.fusefss_debug_set(b"coop", 1) == 0
    assert F.lib.fusefss_prepare(None) == -1
