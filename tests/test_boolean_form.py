"""The Boolean form the kernels use (csrc/xs_device.cuh, a-4..a-7) against the +-1 rule of the
paper, exhaustively over all 2^11 inputs: 6 partner bits, 3 coupling
bits, own bit, noise bit.  The LOP3 truth-table constants are read from the CUDA header, so a
wrong LUT in the product fails here without a GPU."""
from __future__ import annotations

import itertools
import os
import re

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _luts():
    src = open(os.path.join(ROOT, "paper_2102_09510_b200", "csrc", "xs_device.cuh")).read()
    out = {}
    for name in ("LUT_XOR3", "LUT_MAJ", "LUT_MAJ_NOTC", "LUT_SEL", "LUT_NZ"):
        m = re.search(r"constexpr int %s = (0x[0-9A-Fa-f]+);" % name, src)
        assert m, name
        out[name] = int(m.group(1), 16)
    # the order of the lop3 calls in qg_update / qg_nonzero_k is part of what is checked
    assert re.search(r"w0 = lop3<LUT_XOR3>\(a0, b0, j0\)", src)
    assert re.search(r"M = lop3<LUT_MAJ>\(w0, w1, w2\)", src)
    assert re.search(r"P = lop3<LUT_XOR3>\(w0, w1, w2\)", src)
    assert re.search(r"f = lop3<LUT_MAJ_NOTC>\(M, P, x\)", src)
    assert re.search(r"return lop3<LUT_SEL>\(R, f, M\)", src)
    assert re.search(r"return lop3<LUT_NZ>\(M, P, x\)", src)
    return out


def lop3(lut, a, b, c):
    return (lut >> (a * 4 + b * 2 + c)) & 1      # PTX lop3: bit index = a*4 + b*2 + c


def test_boolean_update_equals_pm1_rule_on_all_inputs():
    L = _luts()
    for bits in itertools.product((0, 1), repeat=11):
        a0, b0, a1, b1, a2, b2, j0, j1, j2, x, R = bits
        # +-1 arithmetic: bit 1 <=> spin -1, jbit 1 <=> J = -1
        s = lambda v: 1 - 2 * v                                    # noqa: E731
        k = sum(1 for (a, b, j) in ((a0, b0, j0), (a1, b1, j1), (a2, b2, j2))
                if s(j) * s(x) * s(a) * s(b) == -1)                # unsatisfied interactions
        flip = (k >= 2) or (k == 1 and R == 1)                     # w = (0, w1, 1, 1)
        x_new_ref = x ^ int(flip)
        # Boolean form
        w0, w1, w2 = (lop3(L["LUT_XOR3"], a0, b0, j0), lop3(L["LUT_XOR3"], a1, b1, j1),
                      lop3(L["LUT_XOR3"], a2, b2, j2))
        M, P = lop3(L["LUT_MAJ"], w0, w1, w2), lop3(L["LUT_XOR3"], w0, w1, w2)
        f = lop3(L["LUT_MAJ_NOTC"], M, P, x)
        x_new = lop3(L["LUT_SEL"], R, f, M)
        assert x_new == x_new_ref, bits
        assert lop3(L["LUT_NZ"], M, P, x) == int(k != 0), bits
        assert 2 * (M ^ x) + (P ^ x) == k, bits                    # the bit-sliced adder
        assert 6 - 4 * k in (6, 2, -2, -6)                         # Delta E of the flip (L67)


def _src(name):
    return open(os.path.join(ROOT, "paper_2102_09510_b200", "csrc", name)).read()


def test_clause_word_forms_equal_pm1_rule_on_all_inputs():
    """The clause-word kernels (xs_sweep_clause.cuh, xs_sweep_warp.cu) update from the three clause
    bits c_r = x ^ a_r ^ b_r ^ j_r (1 <=> interaction r unsatisfied, L65-L67): k = c_0 + c_1 + c_2,
    flip iff k >= 2 or (k = 1 and R) (L101), and a flip toggles the spin and its three clauses.
    LUT constants and operand orders are read from the CUDA sources."""
    L = _luts()
    cl = _src("xs_sweep_clause.cuh")
    m = re.search(r"constexpr int LUT_OR_ANDN = (0x[0-9A-Fa-f]+);", cl)
    assert m
    or_andn = int(m.group(1), 16)
    assert re.search(r"M = lop3<LUT_MAJ>\(c0\[c\], c1\[c\], c2\[c\]\)", cl)
    assert re.search(r"P = lop3<LUT_XOR3>\(c0\[c\], c1\[c\], c2\[c\]\)", cl)
    assert re.search(r"lop3<LUT_OR_ANDN>\(M, P, nf\[c >> 1\]\)", cl)          # nf = NOT-flip mask (u >= thr)
    m = re.search(r"f = PCN \? lop3<(0x[0-9A-Fa-f]+)>\(M, P, rc\[c\]\)", cl)     # per-clone noise: rc = flip mask
    assert m
    pcn_lut = int(m.group(1), 16)
    m = re.search(r"if \(W0\) f = lop3<(0x[0-9A-Fa-f]+)>\(f, n0\[c >> 1\], 0u\);", cl)   # n0 = NOT-flip mask of k = 0
    assert m
    w0_lut = int(m.group(1), 16)
    m = re.search(r"lacc\[c\] = lop3<(0x[0-9A-Fa-f]+)>\(c0\[c\], l0, lacc\[c\]\);", cl)
    assert m
    acc_lut = int(m.group(1), 16)
    assert re.search(r"c0\[c\] \^= f; c1\[c\] \^= f; c2\[c\] \^= f;\s*x\[r\]\[c\] \^= f;", cl)
    m = re.search(r"PACK \? lop3<(0x[0-9A-Fa-f]+)>\(nb, rm\[r\], 0x80808080u\) : nb", cl)
    assert m
    merge = int(m.group(1), 16)
    wp = _src("xs_sweep_warp.cu")
    m = re.search(r"constexpr int LUT_OR_AND = (0x[0-9A-Fa-f]+);", wp)
    assert m
    or_and = int(m.group(1), 16)
    assert re.search(r"f = lop3<LUT_OR_AND>\(M, P, R\)", wp)                  # R = flip mask (u < thr)
    assert re.search(r"wp_sts\(ca\[r\]\[0\], c0 \^ f\);\s*wp_sts\(ca\[r\]\[1\], c1 \^ f\);\s*wp_sts\(ca\[r\]\[2\], c2 \^ f\);\s*x\[r\] \^= f;", wp)
    for bits in itertools.product((0, 1), repeat=11):
        a0, b0, a1, b1, a2, b2, j0, j1, j2, x, R = bits
        s = lambda v: 1 - 2 * v                                    # noqa: E731
        unsat = [int(s(j) * s(x) * s(a) * s(b) == -1) for (a, b, j) in ((a0, b0, j0), (a1, b1, j1), (a2, b2, j2))]
        k = sum(unsat)
        flip = int((k >= 2) or (k == 1 and R == 1))
        c = [x ^ a0 ^ b0 ^ j0, x ^ a1 ^ b1 ^ j1, x ^ a2 ^ b2 ^ j2]
        assert c == unsat, bits                                    # clause bit = "unsatisfied"
        # clause-word kernel: threshold bytes hold NOT R
        M, P = lop3(L["LUT_MAJ"], *c), lop3(L["LUT_XOR3"], *c)
        assert lop3(or_andn, M, P, 1 - R) == flip, bits
        assert lop3(pcn_lut, M, P, R) == flip, bits
        # tables (w0, w1, 1, 1), w0 <= w1, one number per word: R0 = (u < thr0) implies R = (u < thr1)
        for R0 in ((0, 1) if R else (0,)):
            flip_w0 = int((k >= 2) or (k == 1 and R == 1) or (k == 0 and R0 == 1))
            assert lop3(w0_lut, lop3(or_andn, M, P, 1 - R), 1 - R0, 0) == flip_w0, bits
        # after the flip the clause bits must be those of the new spin value
        x_new = x ^ flip
        c_new = [x_new ^ a0 ^ b0 ^ j0, x_new ^ a1 ^ b1 ^ j1, x_new ^ a2 ^ b2 ^ j2]
        assert [ci ^ flip for ci in c] == c_new, bits
        # latency kernel: the same with the mask R itself
        assert lop3(or_and, M, P, R) == flip, bits
    for a, b, cc in itertools.product((0, 1), repeat=3):
        assert lop3(acc_lut, a, b, cc) == ((a & b) | cc)              # last-touch accumulate
    # the merge of new threshold bits into the register that also carries the spin index
    for a, b, cc in itertools.product((0, 1), repeat=3):
        assert lop3(merge, a, b, cc) == (a if cc else b)
