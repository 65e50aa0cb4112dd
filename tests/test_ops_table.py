"""A second source for the roofline numerator (VERDICT r01 "missing" 4): the FP64 operation
list of the reduced algorithm (DESIGN.md 5.1 / 6), restated here as a table counted from the formulas, must agree with
what ncu counted on the kernels (profiles/r02_ops.json) to about one per cent -- so that "executed = algorithmic" is
checked, and a kernel change that adds redundant work (or a stale ops file) shows up.

Counting rules: one fma / mul / add each; negations are operand modifiers (free); products that the six brackets
share (sin(theta) E_n, used by two brackets each) are counted once; 2 x and x + x are adds; a product whose only use is
an addition is one fma (nvcc --fmad contracts them: the magic-constant add of the phase reduction, tau into the orbit
angle); anything that depends on the bin and compile-time constants only (ln f + ln(2/m)/3, (m/2)^{8/3} f^{-5/3}) is
hoisted out of the sample loop and is not per-unit work.
"""
import json
import os

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
OPS = os.path.join(ROOT, "profiles", "r02_ops.json")

SINCOS_TAB = {"fma": 6, "mul": 3, "add": 3}          # sincos_tab: split (3 add), y^2, two short polynomials, angle addition


def add_ops(total, ops, times=1):
    for k, v in ops.items():
        total[k] = total.get(k, 0) + times * v


def wave_ops(mc: int):
    """S2/S3 of one mode class (m = mc + 1): eval_class up to the call of eval_geom (pespace_device.cuh)"""
    t = {"fma": 0, "mul": 0, "add": 0}
    if mc != 1:
        add_ops(t, {"mul": 1})                              # v = v_2 (2/m)^{1/3}
    add_ops(t, {"mul": 1})                                  # v^2
    add_ops(t, {"fma": 8 + 7})                              # P (8 incl. the two log terms), Q (7)
    add_ops(t, {"mul": 1, "fma": 1, "add": 2})              # psi = s P; psi -= ((psi + magic) - magic)
    add_ops(t, {"add": 2} if mc == 1 else {"fma": 1, "add": 1})     # + (m/2) PH0 + f t_c
    add_ops(t, {"fma": 2} if mc == 1 else {"mul": 2})       # amplitudes a + b v^2 | v^p a
    return t


def geom_ops(kind: int, tau_cached: bool = False):
    """S4-S7 of one class for one detector: eval_geom.  tau_cached: the fused kernel keeps tau = s' Q in a register,
    the per-detector kernel contracts that product into the orbit-angle sum"""
    t = {"fma": 0, "mul": 0, "add": 0}
    # S4: orbit angle(s) and G1, G2 of k, u', v', Doppler phase of the centre
    if kind == 0:
        add_ops(t, {"add": 1} if tau_cached else {"fma": 1}); add_ops(t, SINCOS_TAB)     # alpha = alpha0 + tau; sin, cos
        add_ops(t, {"fma": 1, "add": 2, "mul": 1})          # cos 2a = 2 c c - 1, sin 2a = (s + s) c
        add_ops(t, {"fma": 18})                             # six three-term combinations
    else:
        add_ops(t, {"add": 1, "fma": 1} if tau_cached else {"mul": 1, "fma": 2}); add_ops(t, SINCOS_TAB, 2)
        add_ops(t, {"fma": 6, "mul": 6})
    add_ops(t, {"fma": 1, "mul": 1})                        # k.R
    # projections: k.delta_n, k.n_l, u'.n_l, v'.n_l with literal coefficients
    add_ops(t, {"mul": 3, "fma": 8, "add": 3})
    # S5: three arm weights (squares, reciprocal = 3 fma after the hardware seed, two products each for + and x)
    add_ops(t, {"mul": 6, "fma": 5}, 3)
    # S6: phase at the centre, three exponentials
    add_ops(t, {"fma": 1})
    add_ops(t, {"fma": 1}, 3); add_ops(t, SINCOS_TAB, 3)
    # S7: six brackets (E_s - cos E_r, kap x, +- sin E_r) and W.B products; sin(theta) E_n shared by two brackets
    add_ops(t, {"fma": 4}, 6)
    add_ops(t, {"mul": 6})                                  # sin(theta) (Er, Ei)[n], n = 1..3
    add_ops(t, {"fma": 4}, 6)                               # complex W B accumulated (first class: 2 fma + 2 mul)
    return t


FIRST_CLASS = {"fma": -6, "mul": 6}                         # initialising S: 2 fma + 2 mul instead of 4 fma, x 3
RESIDUAL = {"add": 2 + 2 + 4 + 6, "fma": 2 + 5, "mul": 4}   # A, E, T, residuals, weighted squares


def loglike_ops(classes, kind, single_class):
    """loglike_kernel<kind, mask>: per (sample, bin) of ONE detector"""
    t = {"fma": 0, "mul": 0, "add": 0}
    add_ops(t, {"mul": 2, "add": 2, "fma": 1})              # f t_c modulo one turn, v = a f^{1/3}
    for i, mc in enumerate(classes):
        add_ops(t, wave_ops(mc)); add_ops(t, geom_ops(kind))
        if i == 0:
            add_ops(t, FIRST_CLASS)
    add_ops(t, RESIDUAL)
    add_ops(t, {"add": 1.5 if single_class else 5.0})       # warp reduction per unit
    return t


def fused_ops(classes, kinds):
    """loglike_fused_kernel<mask>: per (sample, bin, detector), averaged over the detectors of the model: the waveform
    part once per (sample, bin), S4-S8 per detector, one reduction per (sample, bin)"""
    t = {"fma": 0, "mul": 0, "add": 0}
    add_ops(t, {"mul": 2, "add": 2, "fma": 1})
    for mc in classes:
        add_ops(t, wave_ops(mc)); add_ops(t, {"mul": 1})    # + tau kept as a product of its own
    for kind in kinds:
        for i, mc in enumerate(classes):
            add_ops(t, geom_ops(kind, tau_cached=True))
            if i == 0:
                add_ops(t, FIRST_CLASS)
        add_ops(t, RESIDUAL)
    add_ops(t, {"add": 5.0})
    return {k: v / len(kinds) for k, v in t.items()}


@pytest.fixture(scope="module")
def ops():
    assert os.path.exists(OPS), "profiles/r02_ops.json is missing (python -m paper_2602_12011_b200.ops_from_ncu)"
    return json.load(open(OPS))


@pytest.mark.parametrize("key,classes,kind", [("loglike|0|2", [1], 0), ("loglike|0|15", [0, 1, 2, 3], 0),
                                               ("loglike_fused|0|15", [0, 1, 2, 3], (0, 0, 1))])
def test_operation_table_sums_to_the_ncu_count(ops, key, classes, kind):
    """config 2 (one class, LISA-like), config 3 (four classes, LISA-like), config 4 (four classes, two heliocentric
    detectors and a geocentric one in the fused kernel)"""
    row = ops["kernels"].get(key)
    assert row is not None, key
    t = fused_ops(classes, kind) if isinstance(kind, tuple) else loglike_ops(classes, kind, single_class=len(classes) == 1)
    want = sum(t.values())
    got = row["dfma"] + row["dmul"] + row["dadd"]
    assert abs(got - want) <= 0.015 * got, (key, t, row["dfma"], row["dmul"], row["dadd"])
    assert abs(t["fma"] - row["dfma"]) <= 0.02 * row["dfma"], (t["fma"], row["dfma"])
    flop = 2 * t["fma"] + t["mul"] + t["add"]
    assert abs(flop - row["flop_per_unit"]) <= 0.015 * row["flop_per_unit"]


def test_ops_file_is_stamped(ops):
    from paper_2602_12011_b200 import build
    assert isinstance(ops.get("csrc_hash"), str) and len(ops["csrc_hash"]) == 16
    assert ops["unit"] == "(sample, bin, detector)"
    # not asserted equal to build.csrc_hash(): bench.py reports roofline.stale when the kernels moved on
    assert len(build.csrc_hash()) == 16


def test_kernel_names_map_to_table_keys():
    """ops_from_ncu.kernel_key: demangled ncu kernel names -> (kernel, kind, class mask) of the table keys bench.py reads"""
    from paper_2602_12011_b200.ops_from_ncu import kernel_key
    assert kernel_key("void pespace::loglike_kernel<0, 2>(const double *, ...)") == ("loglike", 0, 2)
    assert kernel_key("void pespace::loglike_kernel<1, 15u>(const double *)") == ("loglike", 1, 15)
    assert kernel_key("void pespace::loglike_fused_kernel<15>(const double *)") == ("loglike_fused", 0, 15)
    assert kernel_key("void pespace::response_fused_kernel<15u>(const double *)") == ("response_fused", 0, 15)
    assert kernel_key("void pespace::response_kernel<0, 2>(const double *)") == ("response", 0, 2)
    assert kernel_key("void pespace::loglike_orb_kernel<2>(const double *)") == ("loglike_orb", 0, 2)
    assert kernel_key("void pespace::loglike_tab_kernel<0, 5>(const double *)") == ("loglike_tab", 0, 5)
    assert kernel_key("void pespace::fisher_kernel<1, 15>(const double *)") == ("fisher", 1, 15)
    assert kernel_key("void pespace::combine_kernel(const double *)") is None
