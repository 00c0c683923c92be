"""DESIGN.md section 4, tolerance T, checked in numpy (no GPU, no library): the fp32 arithmetic the kernels use for one
output x*c + y*t -- restated here with float32 arrays, an FMA being one rounding of the exact fp64 product-sum -- against
the exact value rounded once to bf16 (what the oracle stores).

  * the plain form alone (round 1) is within one bf16 code wherever |r| >= 2^-12 |p|, and is many codes off on results
    that cancel deeper: the reason the rule exists;
  * the rule (plain, and the compensated form where |r| < 2^-12 |p|) is within ONE code everywhere, so that the test
    bar "<= 2 bf16 ulp for every element, no cancellation floor" (tests/parity.py) has a margin of one.
"""
import numpy as np

F = np.float32


def fma32(a, b, c):
    """One rounding of a*b + c: the product of two fp32 values is exact in fp64 (48 bits), the sum is rounded to fp64 and
    then to fp32 (a double rounding that matters once in ~2^29 cases: irrelevant for a statement about bf16 codes)."""
    return (a.astype(np.float64) * b.astype(np.float64) + c.astype(np.float64)).astype(F)


def rot_plain(x, ch, y, th):
    p = (x * ch).astype(F)
    return fma32(y, th, p), p


def rot_comp(x, ch, cl, y, th, tl):
    q = (y * th).astype(F)
    e = fma32(y, th, -q)                       # exact: the rounding error of q
    r1 = fma32(x, ch, q)
    return (r1 + fma32(x, cl, fma32(y, tl, e))).astype(F)


def bf16_code(v64):
    """Ordinal of the bf16 value nearest (RNE) to v: sign-magnitude codes mapped to a line."""
    f = np.asarray(v64, np.float64).astype(F)            # inputs here are fp32-representable or rounded once below
    u = f.view(np.uint32).astype(np.uint64)
    u = (u + 0x7FFF + ((u >> 16) & 1)) >> 16               # RNE of the top 16 bits
    mag = (u & 0x7FFF).astype(np.int64)
    return np.where(u & 0x8000, -mag, mag)


def bf16_code_exact(v64):
    """Code of the fp64 value rounded ONCE to bf16 (the oracle's direct rounding): through a 24-bit-safe path -- bf16 has
    8 significant bits, so rounding the fp64 value to fp32 first can only matter at exact ties of the 16 dropped bits,
    which round-to-odd on the way removes."""
    v = np.asarray(v64, np.float64)
    f = v.astype(F)
    # round-to-odd fp64 -> fp32: if inexact, force the last bit to 1 so that the second rounding cannot hit a false tie
    inexact = f.astype(np.float64) != v
    bits = f.view(np.uint32)
    toward_zero = np.where(np.abs(f.astype(np.float64)) > np.abs(v), bits - 1, bits)
    bits = np.where(inexact, toward_zero | 1, bits).astype(np.uint32)
    return bf16_code(bits.view(F).astype(np.float64))


def make_inputs(rng, n, deep):
    """bf16-representable pairs (a, b) and angles; `deep`: a is chosen so that a cos - b sin nearly cancels."""
    phi = rng.uniform(-np.pi, np.pi, n)
    c64, s64 = np.cos(phi), np.sin(phi)
    b = (rng.standard_normal(n) * 2).astype(F)
    a = (b.astype(np.float64) * s64 / np.where(np.abs(c64) < 0.05, 0.05, c64)).astype(F) if deep else (rng.standard_normal(n) * 2).astype(F)
    to_bf16 = lambda v: ((v.view(np.uint32) + 0x7FFF + ((v.view(np.uint32) >> 16) & 1)) & 0xFFFF0000).astype(np.uint32).view(F)
    return to_bf16(a), to_bf16(b), c64, s64


def kernel_rule(a, b, c64, s64):
    ch, sh = c64.astype(F), s64.astype(F)
    cl, sl = (c64 - ch.astype(np.float64)).astype(F), (s64 - sh.astype(np.float64)).astype(F)
    r, p = rot_plain(a, ch, b, -sh)
    fix = np.abs(r) * F(4096.0) < np.abs(p)
    return np.where(fix, rot_comp(a, ch, cl, b, -sh, -sl), r), r, fix


def test_plain_form_needs_the_fix_up_and_the_rule_is_within_one_code():
    rng = np.random.default_rng(7)
    worst_rule, worst_plain, n_fix = 0, 0, 0
    for deep in (False, True):
        a, b, c64, s64 = make_inputs(rng, 2_000_000, deep)
        exact = a.astype(np.float64) * c64 - b.astype(np.float64) * s64
        want = bf16_code_exact(exact)
        got, plain, fix = kernel_rule(a, b, c64, s64)
        d_rule = np.abs(bf16_code(got.astype(np.float64)) - want)
        d_plain = np.abs(bf16_code(plain.astype(np.float64)) - want)
        assert d_rule.max() <= 1, f"the rule is {int(d_rule.max())} codes off (deep={deep})"
        assert d_plain[~fix].max() <= 1            # where the rule keeps the plain form, the plain form is enough
        worst_rule, worst_plain, n_fix = max(worst_rule, int(d_rule.max())), max(worst_plain, int(d_plain.max())), n_fix + int(fix.sum())
    assert n_fix > 1000                            # the constructed inputs do exercise the compensated form ...
    assert worst_plain > 2                         # ... on which the plain form alone would break the 2-ulp bar


def test_compensated_form_is_accurate_to_fp32_relative_precision():
    rng = np.random.default_rng(8)
    a, b, c64, s64 = make_inputs(rng, 1_000_000, True)
    ch, sh = c64.astype(F), s64.astype(F)
    cl, sl = (c64 - ch.astype(np.float64)).astype(F), (s64 - sh.astype(np.float64)).astype(F)
    exact = a.astype(np.float64) * c64 - b.astype(np.float64) * s64
    got = rot_comp(a, ch, cl, b, -sh, -sl).astype(np.float64)
    rho = np.hypot(a.astype(np.float64), b.astype(np.float64))
    err = np.abs(got - exact)
    assert (err <= 2.0 ** -23 * np.abs(exact) + 2.0 ** -44 * rho).all()     # ~2^-24 |r| + 2^-47 rho, with a factor to spare
    plain = rot_plain(a, ch, b, -sh)[0].astype(np.float64)
    assert (np.abs(plain - exact) <= 1.7 * 2.0 ** -24 * 1.5 * rho + 1e-300).all()   # the plain form's ABSOLUTE bound
    assert (np.abs(plain - exact) > 2.0 ** -20 * np.abs(exact)).any()           # ... which is not a relative one
