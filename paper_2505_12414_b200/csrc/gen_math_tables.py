"""Generates mf_math_tables.inc: polynomial coefficients and the log table of mf_math.cuh.

    python paper_2505_12414_b200/csrc/gen_math_tables.py

Everything is computed here with mpmath at 80 digits and rounded once to double:
  * exp(r) ~ 1 + r + r^2 q(r) on |r| <= ln2/2 (1 + 2^-20): q of degree 9 interpolated at
    Chebyshev nodes of (exp(r) - 1 - r)/r^2 (near-minimax);
  * log1p(rho) ~ rho + rho^2 q(rho) on |rho| <= 2^-7.9: q of degree 4, same construction;
  * the 128-entry log table: for m in [sqrt(1/2), sqrt(2)) the index is bits of the high word,
    j = ((hi(m) - 0x3fe6a09e) >> 13) & 127; entry j holds invc_j = fl(1/c_j) and
    logc_j = fl(-log(invc_j)), c_j the interval midpoint (c = 1 exactly for the interval that
    contains 1, so log is exact to rounding near 1).
The script prints the achieved approximation errors; mf_math.cuh states them.
"""
import os
import struct

import mpmath as mp

mp.mp.dps = 80
OFF = 0x3FE6A09E


def to_double(x) -> float:
    return float(mp.nstr(x, 40))


def hexlit(d: float) -> str:
    return float(d).hex()


def cheb_fit(f, a, b, deg):
    """Polynomial of degree `deg` interpolating f at the deg+1 Chebyshev nodes of [a, b]; monomial coefficients."""
    n = deg + 1
    xs = [(a + b) / 2 + (b - a) / 2 * mp.cos(mp.pi * (2 * k + 1) / (2 * n)) for k in range(n)]
    A = mp.matrix(n, n)
    y = mp.matrix(n, 1)
    for i, x in enumerate(xs):
        for j in range(n):
            A[i, j] = x ** j
        y[i] = f(x)
    c = mp.lu_solve(A, y)
    return [c[j] for j in range(n)]


def horner(cs, x):
    s = mp.mpf(0)
    for c in reversed(cs):
        s = s * x + c
    return s


def max_err(approx, exact, a, b, n=4001, rel=True):
    worst = mp.mpf(0)
    for k in range(n):
        x = a + (b - a) * k / (n - 1)
        if x == 0:
            continue
        e = abs(approx(x) - exact(x))
        if rel:
            e /= abs(exact(x))
        worst = max(worst, e)
    return worst


def dbl_from_hi(hi: int) -> float:
    return struct.unpack("<d", struct.pack("<II", 0, hi))[0]


def main():
    out = []
    # ---- exp
    R = mp.log(2) / 2 * (1 + mp.mpf(2) ** -20)
    q_exp = cheb_fit(lambda r: (mp.exp(r) - 1 - r) / r ** 2 if abs(r) > mp.mpf(10) ** -30 else mp.mpf(1) / 2 + r / 6, -R, R, 9)
    q_exp_d = [to_double(c) for c in q_exp]
    err = max_err(lambda r: 1 + r + r * r * horner([mp.mpf(c) for c in q_exp_d], r), mp.exp, -R, R)
    print(f"exp: degree-11 relative error with double coefficients = {mp.nstr(err, 4)}")
    out.append("// exp(r) = 1 + r + r^2 (c[0] + c[1] r + ... + c[9] r^9) on |r| <= ln2/2; max rel. error %s" % mp.nstr(err, 3))
    out.append("#define MF_EXP_POLY { " + ", ".join(hexlit(c) for c in q_exp_d) + " }")
    # ---- exp with a 32-entry table: exp(x) = 2^e 2^(j/32) exp(r), |r| <= ln2/64
    R32 = mp.log(2) / 64 * (1 + mp.mpf(2) ** -12)
    q32 = cheb_fit(lambda r: (mp.exp(r) - 1 - r) / r ** 2 if abs(r) > mp.mpf(10) ** -30 else mp.mpf(1) / 2 + r / 6, -R32, R32, 4)
    q32_d = [to_double(c) for c in q32]
    err = max_err(lambda r: 1 + r + r * r * horner([mp.mpf(c) for c in q32_d], r), mp.exp, -R32, R32)
    print(f"exp32: degree-6 relative error with double coefficients = {mp.nstr(err, 4)}")
    assert err < mp.mpf(2) ** -58
    out.append("// exp(r) - 1 = r + r^2 (c[0] + ... + c[4] r^4) on |r| <= ln2/64; max rel. error of exp %s" % mp.nstr(err, 3))
    out.append("#define MF_EXP32_POLY { " + ", ".join(hexlit(c) for c in q32_d) + " }")
    out.append("// 2^(j/32), j = 0..31, rounded to nearest")
    out.append("#define MF_EXP2_32_TABLE { " + ", ".join(hexlit(to_double(mp.mpf(2) ** (mp.mpf(j) / 32))) for j in range(32)) + " }")
    # ---- log1p on the table residual
    lo_hi = []
    tab = []
    worst_rho = mp.mpf(0)
    for j in range(128):
        a = mp.mpf(dbl_from_hi(OFF + j * 8192))
        b = mp.mpf(dbl_from_hi(OFF + (j + 1) * 8192))
        c = mp.mpf(1) if a <= 1 < b else (a + b) / 2
        invc = to_double(1 / c)
        logc = to_double(-mp.log(mp.mpf(invc)))
        tab.append((invc, logc))
        worst_rho = max(worst_rho, abs(a * mp.mpf(invc) - 1), abs(b * mp.mpf(invc) - 1))
        lo_hi.append((a, b))
    print(f"log: max |rho| = 2^{mp.nstr(mp.log(worst_rho, 2), 5)}")
    assert worst_rho < mp.mpf(2) ** -7.9
    Q = worst_rho * (1 + mp.mpf(2) ** -10)
    q_log = cheb_fit(lambda r: (mp.log1p(r) - r) / r ** 2 if abs(r) > mp.mpf(10) ** -30 else -mp.mpf(1) / 2 + r / 3, -Q, Q, 4)
    q_log_d = [to_double(c) for c in q_log]
    err = max_err(lambda r: r + r * r * horner([mp.mpf(c) for c in q_log_d], r), mp.log1p, -Q, Q)
    print(f"log1p: degree-6 relative error with double coefficients = {mp.nstr(err, 4)}")
    out.append("// log1p(rho) = rho + rho^2 (c[0] + ... + c[4] rho^4) on |rho| <= %s; max rel. error %s"
               % (mp.nstr(Q, 4), mp.nstr(err, 3)))
    out.append("#define MF_LOG1P_POLY { " + ", ".join(hexlit(c) for c in q_log_d) + " }")
    out.append("// {invc_j, logc_j}: m * invc_j - 1 = rho, log(m) = logc_j + log1p(rho)")
    out.append("#define MF_LOG_TABLE { \\")
    for invc, logc in tab:
        out.append("    {%s, %s}, \\" % (hexlit(invc), hexlit(logc)))
    out.append("}")
    ln2 = mp.log(2)
    ln2_hi = float(int(ln2 * 2 ** 42) / 2 ** 42)            # 42 significant bits: n * ln2_hi is exact for |n| < 2^11
    ln2_lo = to_double(ln2 - mp.mpf(ln2_hi))
    out.append("#define MF_LN2_HI %s" % hexlit(ln2_hi))
    out.append("#define MF_LN2_LO %s" % hexlit(ln2_lo))
    out.append("#define MF_LN2 %s" % hexlit(to_double(ln2)))
    out.append("#define MF_LOG2E %s" % hexlit(to_double(1 / ln2)))
    path = os.path.join(os.path.dirname(os.path.abspath(__file__)), "mf_math_tables.inc")
    with open(path, "w") as fh:
        fh.write("// GENERATED by gen_math_tables.py (mpmath, 80 digits) — do not edit.\n")
        fh.write("\n".join(out) + "\n")
    print("wrote", path)


if __name__ == "__main__":
    main()
