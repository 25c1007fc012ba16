"""Derives the polynomial coefficients of csrc/trig.cuh (sincos_cw, exp_cw) by a Remez exchange in 60-digit arithmetic.

    python paper_1601_04640_b200/csrc/trig_coefficients.py

sin r = r + r^3 P(r^2) and cos r = 1 - r^2/2 + r^4 Q(r^2) on |r| <= pi/4 (P, Q of degree 5 in r^2), and
exp r = 1 + r + r^2 E(r) on |r| <= ln(2)/2 (E of degree 9); P and Q minimise the maximum ABSOLUTE error of the
function, E its own (the error of exp is that times r^2 <= 0.12).  Prints the error bounds and the coefficients as decimal doubles (lowest power first).  The numbers in
trig.cuh are this script's output; tests/test_host_logic.py pins the finished functions against long-double libm.
"""
import mpmath as mp

mp.mp.dps = 60


def remez(f, deg, weight, lo, hi, iters=14, grid=4000):
    """Coefficients c[0..deg] minimising max |weight(x) (f(x) - sum c_j x^j)| on [lo, hi]."""
    n = deg + 2
    xs = [lo + (hi - lo) * (1 - mp.cos(mp.pi * k / (n - 1))) / 2 for k in range(n)]
    c, worst = None, None
    for _ in range(iters):
        A, b = mp.matrix(n, n), mp.matrix(n, 1)
        for i, x in enumerate(xs):
            for j in range(deg + 1):
                A[i, j] = x ** j
            A[i, deg + 1] = (-1) ** i / weight(x)
            b[i] = f(x)
        sol = mp.lu_solve(A, b)
        c = [sol[j] for j in range(deg + 1)]
        pts = [lo + (hi - lo) * k / grid for k in range(grid + 1)]
        vals = [weight(p) * (f(p) - sum(c[j] * p ** j for j in range(deg + 1))) for p in pts]
        worst = max(abs(v) for v in vals)
        ext = []
        for k, v in enumerate(vals):
            left = vals[k - 1] if k > 0 else None
            right = vals[k + 1] if k < grid else None
            if (left is None or abs(v) >= abs(left)) and (right is None or abs(v) >= abs(right)):
                if not ext or (v > 0) != (ext[-1][1] > 0):
                    ext.append((pts[k], v))
                elif abs(v) > abs(ext[-1][1]):
                    ext[-1] = (pts[k], v)
        while len(ext) > n:
            ext.pop(0) if abs(ext[0][1]) < abs(ext[-1][1]) else ext.pop()
        if len(ext) == n:
            xs = [e[0] for e in ext]
    return c, worst


def main():
    tiny = mp.mpf(10) ** -40
    T = (mp.pi / 4) ** 2

    def fP(t):
        r = mp.sqrt(t)
        return -mp.mpf(1) / 6 if t == 0 else (mp.sin(r) - r) / r ** 3

    def fQ(t):
        r = mp.sqrt(t)
        return mp.mpf(1) / 24 if t == 0 else (mp.cos(r) - 1 + t / 2) / t ** 2

    a = mp.log(2) / 2

    def fE(r):
        if abs(r) < mp.mpf(10) ** -15:                     # (the middle node is 0 up to rounding: no cancellation there)
            return mp.mpf(1) / 2 + r / 6 + r * r / 24
        return (mp.exp(r) - 1 - r) / r ** 2

    for name, f, deg, w, lo, hi in (("sin: P (r^3 .. r^13)", fP, 5, lambda t: t ** mp.mpf(1.5) if t > 0 else tiny, 0, T),
                                    ("cos: Q (r^4 .. r^14)", fQ, 5, lambda t: t ** 2 if t > 0 else tiny, 0, T),
                                    ("exp: E (r^2 .. r^11)", fE, 9, lambda r: mp.mpf(1), -a, a)):
        c, err = remez(f, deg, w, lo, hi)
        print(f"{name}: max absolute error {mp.nstr(err, 4)}")
        for x in c:
            print("   ", repr(float(x)))


if __name__ == "__main__":
    main()
