"""Generates paper_2606_17065_b200/csrc/coeffs.cuh: polynomial coefficients of the device special functions.

Build-step script (run by hand when an approximation changes; the generated header is committed so that building
the library needs only nvcc).  Everything is derived here from mpmath at 40 digits -- no published coefficient table
is used, and nothing is shared with oracle/ (which uses libm in long double).

  erfcx(z), z >= ZMIN (fp64):  y = (z - C)/(z + C),  erfcx(z) = (1 - y) Q(y),  Q = degree-N polynomial in y on
                            [y(ZMIN), 1] (Chebyshev interpolant converted to the monomial basis; (1-y) = 2C/(z+C) keeps the
                            1/z decay exact, so Q is smooth up to y = 1 <=> z = infinity).  ZMIN = -0.0708 is slightly
                            negative and the degree is chosen for the DERIVATIVE of Q as well: the solver forms
                            erfcx(z1) - erfcx(z2) from the divided difference Q[y1, y2] (lbr_device.cuh, erfcx_dd), whose
                            error is that of Q' (Markov: up to N^2 times the error of Q near the ends of the interval)
  erfcx(z), z >= ZMIN (fp32):  same form, lower degree, for the seed (needs ~1e-6)
  Phi^-1 tail (fp32):       for p <= 1/2 with u = sqrt(-2 ln p):  -Phi^-1(p) = u - R(u), R = polynomial in w = 1/(1+u)
                            ... fitted by least squares on Chebyshev nodes (seed accuracy ~1e-5 relative)
Prints the achieved accuracies; writes the header next to this file.
"""
import os

import mpmath as mp
import numpy as np

mp.mp.dps = 40
HERE = os.path.dirname(os.path.abspath(__file__))


def erfcx(z):
    z = mp.mpf(z)
    return mp.exp(z * z) * mp.erfc(z)


def cheb_coeffs(f, N):
    xs = [mp.cos(mp.pi * (mp.mpf(i) + mp.mpf(1) / 2) / (N + 1)) for i in range(N + 1)]
    fs = [f(x) for x in xs]
    c = []
    for j in range(N + 1):
        s = mp.mpf(0)
        for i in range(N + 1):
            s += fs[i] * mp.cos(mp.pi * j * (mp.mpf(i) + mp.mpf(1) / 2) / (N + 1))
        c.append(2 * s / (N + 1))
    c[0] /= 2
    return c


def cheb_to_monomial(c):
    """sum_j c_j T_j(y) -> sum_k a_k y^k, exactly in mpmath."""
    N = len(c) - 1
    T = [[mp.mpf(1)], [mp.mpf(0), mp.mpf(1)]]
    for j in range(2, N + 1):
        nxt = [mp.mpf(0)] + [2 * v for v in T[j - 1]]
        for k, v in enumerate(T[j - 2]):
            nxt[k] -= v
        T.append(nxt)
    a = [mp.mpf(0)] * (N + 1)
    for j in range(N + 1):
        for k, v in enumerate(T[j]):
            a[k] += c[j] * v
    return a


ZMIN = -0.0708   # z1 = (|h| - t)/sqrt2 >= -0.1/sqrt2 wherever the difference form is used (lbr_device.cuh, eval_W)


def erfcx_Q(y, C):
    if y >= 1:
        return 1 / (2 * C * mp.sqrt(mp.pi))
    z = C * (1 + y) / (1 - y)
    return erfcx(z) * (z + C) / (2 * C)


def fit_erfcx(C, N, zmin=ZMIN):
    """Q on y in [ymin, 1], ymin = y(zmin): Chebyshev interpolant in u = (y - mid)/half, converted to monomials in y."""
    import math
    ymin = (mp.mpf(zmin) - C) / (mp.mpf(zmin) + C)
    half, mid = (1 - ymin) / 2, (1 + ymin) / 2
    au = cheb_to_monomial(cheb_coeffs(lambda u: erfcx_Q(mid + half * u, C), N))
    out = [mp.mpf(0)] * (N + 1)
    for k, ck in enumerate(au):
        for j in range(k + 1):
            out[j] += ck * math.comb(k, j) * (1 / half) ** k * (-mid) ** (k - j)
    return out


def check_bracket(a, C, zmin=ZMIN):
    """max relative truncation error of Q(y) - (1 - y) Q'(y) (= -erfcx'(z) (z + C)^2 / 2C: what the divided-difference form
    of erfcx(z1) - erfcx(z2) multiplies) over z >= zmin, in mpmath (no rounding)."""
    N = len(a) - 1
    y0 = float((mp.mpf(zmin) - C) / (mp.mpf(zmin) + C))
    worst = 0.0
    for y in np.concatenate([np.linspace(y0, -0.9, 60), np.linspace(-0.9, 0.9995, 120)]):
        ym = mp.mpf(float(y))
        q = sum(a[k] * ym ** k for k in range(N + 1))
        dq = sum(k * a[k] * ym ** (k - 1) for k in range(1, N + 1))
        qt = erfcx_Q(ym, C)
        dqt = mp.diff(lambda t: erfcx_Q(t, C), ym)
        worst = max(worst, abs(float((q - (1 - ym) * dq) / (qt - (1 - ym) * dqt) - 1)))
    return worst


def horner(a, y, dtype):
    acc = dtype(a[-1])
    for v in reversed(a[:-1]):
        acc = dtype(acc * y + dtype(v))
    return acc


def check_erfcx(a, C, dtype):
    zs = np.concatenate([np.linspace(ZMIN, 0, 30), np.linspace(0, 1, 301), np.linspace(1, 12, 1101), np.linspace(12, 60, 200), [1e3, 1e6]])
    worst = 0.0
    af = [dtype(float(v)) for v in a]
    for z in zs:
        z = dtype(z)
        r = dtype(1) / (z + dtype(C))
        y = dtype((z - dtype(C)) * r)
        val = dtype(dtype(2 * C) * r) * horner(af, y, dtype)
        ref = erfcx(mp.mpf(float(z)))
        worst = max(worst, abs(float(mp.mpf(float(val)) / ref - 1)))
    return worst


def fit_ninv_tail(deg):
    """-Phi^-1(p) = u - R(w), u = sqrt(-2 ln p), w = 1/(1+u), p in (0, 0.345]; least squares in w on a dense grid."""
    us = np.concatenate([np.linspace(1.45, 6, 400), np.linspace(6, 40, 300)])   # z >= 0.4 (p <= 0.345): all the seeds need
    zs = []
    for u in us:
        lp = -mp.mpf(u) ** 2 / 2
        # solve ln Phi(-z) = lp by Newton in mpmath
        z = mp.mpf(u)
        for _ in range(60):
            Ph = mp.erfc(z / mp.sqrt(2)) / 2
            ph = mp.exp(-z * z / 2) / mp.sqrt(2 * mp.pi)
            dz = (mp.log(Ph) - lp) * Ph / ph
            z += dz
            if abs(dz) < mp.mpf(10) ** -30:
                break
        zs.append(float(z))
    zs = np.array(zs)
    w = 1.0 / (1.0 + us)
    target = us - zs                                   # R(w)
    A = np.vander(w, deg + 1, increasing=True)
    wt = 1.0 / zs                                      # relative error in z
    coef, *_ = np.linalg.lstsq(A * wt[:, None], target * wt, rcond=None)
    fit = (A @ coef).astype(np.float32)
    rel = np.abs((us.astype(np.float32) - fit) / zs - 1)
    return coef, float(rel.max())



def fit_exp(N):
    """exp(r) on |r| <= ln2/2 as a degree-N polynomial in r (Chebyshev interpolant, monomial basis)."""
    half = mp.log(2) / 2
    a = cheb_to_monomial(cheb_coeffs(lambda y: mp.exp(half * y), N))
    a = [v / half ** k for k, v in enumerate(a)]
    worst = 0.0
    for r in np.linspace(-float(half), float(half), 2001):
        val = horner([float(v) for v in a], np.float64(r), np.float64)
        worst = max(worst, abs(float(mp.mpf(float(val)) / mp.exp(mp.mpf(float(r))) - 1)))
    return a, worst


def fit_atanh(N, fmax):
    """atanh(f) = f (1 + w G(w)), w = f^2 <= fmax^2;  G = degree-N polynomial in w."""
    wmax = mp.mpf(fmax) ** 2

    def G(y):
        w = wmax * (1 + y) / 2
        if w < mp.mpf(10) ** -30:
            return mp.mpf(1) / 3
        f = mp.sqrt(w)
        return (mp.atanh(f) / f - 1) / w
    a = cheb_to_monomial(cheb_coeffs(G, N))
    # y = 2 w / wmax - 1  ->  monomial in w
    out = [mp.mpf(0)] * (N + 1)
    import math
    for k, ck in enumerate(a):
        for j in range(k + 1):
            out[j] += ck * math.comb(k, j) * (2 / wmax) ** j * (-1) ** (k - j)
    worst = 0.0
    for f in np.linspace(1e-6, float(fmax), 1001):
        w = np.float64(f) ** 2
        val = np.float64(f) * (1 + w * horner([float(v) for v in out], w, np.float64))
        worst = max(worst, abs(float(mp.mpf(float(val)) / mp.atanh(mp.mpf(float(f))) - 1)))
    return out, worst

def fmt(vals, per_line=3, f32=False):
    out = []
    for i in range(0, len(vals), per_line):
        chunk = vals[i:i + per_line]
        out.append("    " + ", ".join((f"{float(v):.9e}f" if f32 else f"{mp.nstr(mp.mpf(v), 20, min_fixed=0, max_fixed=0)}") for v in chunk))
    return ",\n".join(out)


def main():
    C64, N64 = 4.0, 24
    a64 = fit_erfcx(C64, N64)
    e64 = check_erfcx(a64, C64, np.float64)
    b64 = check_bracket(a64, C64)
    C32, N32 = 2.0, 10
    a32 = fit_erfcx(C32, N32)
    e32 = check_erfcx(a32, C32, np.float32)
    b32 = check_bracket(a32, C32)
    ninv, en = fit_ninv_tail(7)
    print(f"erfcx fp64: C={C64} N={N64} z >= {ZMIN}: max rel err (fp64 Horner, no FMA) = {e64:.3e}; Q - (1-y)Q' truncation = {b64:.3e}")
    print(f"erfcx fp32: C={C32} N={N32} z >= {ZMIN}: max rel err (fp32 Horner) = {e32:.3e}; Q - (1-y)Q' truncation = {b32:.3e}")
    print(f"ninv tail : deg 7 in w=1/(1+u), max rel err = {en:.3e}")
    NEXP, NATH = 11, 6
    aexp, eexp = fit_exp(NEXP)
    FMAX = (mp.sqrt(2) - 1) / (mp.sqrt(2) + 1) * mp.mpf("1.02")
    aath, eath = fit_atanh(NATH, FMAX)
    print(f"exp       : degree {NEXP} on |r| <= ln2/2, max rel err (fp64 Horner) = {eexp:.3e}")
    print(f"atanh     : f(1 + w G(w)), G degree {NATH}, |f| <= {float(FMAX):.4f}, max rel err = {eath:.3e}")
    with open(os.path.join(HERE, "coeffs.cuh"), "w") as f:
        f.write("// coeffs.cuh -- GENERATED by gen_coeffs.py (mpmath, 40 digits); do not edit by hand.\n")
        f.write(f"// erfcx fp64: erfcx(z) = (2C/(z+C)) Q((z-C)/(z+C)), z >= {ZMIN}, C = {C64}, degree {N64}, max rel err {e64:.2e}; "
                f"Q - (1-y)Q' (divided-difference form) {b64:.2e}\n")
        f.write(f"// erfcx fp32: same form, C = {C32}, degree {N32}, max rel err {e32:.2e}; Q - (1-y)Q' {b32:.2e}\n")
        f.write(f"// ninv tail : -Phi^-1(p) = u - R(1/(1+u)), u = sqrt(-2 ln p), p <= 0.345 (z >= 0.4), degree 7, max rel err {en:.2e}\n")
        f.write(f"// exp       : degree {NEXP} polynomial on |r| <= ln2/2, max rel err {eexp:.2e}\n")
        f.write(f"// atanh     : atanh(f) = f (1 + w G(w)), w = f^2, G degree {NATH}, |f| <= {float(FMAX):.4f}, max rel err {eath:.2e}\n")
        f.write("#pragma once\nnamespace pivot {\n")
        f.write(f"constexpr int kExpN = {NEXP};\n")
        f.write("static __constant__ double kExpP[kExpN + 1] = {\n" + fmt(aexp) + "};\n")
        f.write(f"constexpr int kAtanhN = {NATH};\n")
        f.write("static __constant__ double kAtanhG[kAtanhN + 1] = {\n" + fmt(aath) + "};\n")
        f.write(f"constexpr double kErfcxZmin = {ZMIN};   // the erfcx forms are fitted for z >= kErfcxZmin\n")
        f.write(f"constexpr double kErfcxC = {C64};\nconstexpr int kErfcxN = {N64};\n")
        f.write("static __constant__ __align__(16) double kErfcxQ[kErfcxN + 1] = {\n" + fmt(a64) + "};\n")
        f.write(f"constexpr float kErfcxCf = {C32}f;\nconstexpr int kErfcxNf = {N32};\n")
        f.write("__device__ constexpr float kErfcxQf[kErfcxNf + 1] = {\n" + fmt(a32, 4, True) + "};\n")
        f.write("constexpr int kNinvN = 7;\n")
        f.write("__device__ constexpr float kNinvR[kNinvN + 1] = {\n" + fmt(list(ninv), 4, True) + "};\n")
        f.write("}  // namespace pivot\n")


if __name__ == "__main__":
    main()
