"""Derive the 6th-order symmetric-composition weights used by oracle/aw_oracle.cpp (TEST INFRASTRUCTURE).

The paper (ref. 25 = Yoshida 1990) names a "sixth-order symplectic integrator" but prints
no coefficients.  A 7-stage palindromic composition g = (w3, w2, w1, w0, w1, w2, w3) of a symmetric
2nd-order map is 6th order iff (R2):

    sum g_i = 1,   sum g_i^3 = 0,   sum g_i^5 = 0,
    sum_i g_i^3 * (sum_{j<i} g_j + g_i/2)^2 = 0.

This script solves the four equations with mpmath Newton iteration from the 4-digit neighbourhood of
Yoshida's "solution A" and prints 20 digits.  Run:  python oracle/derive_yoshida6.py
"""
import mpmath as mp

mp.mp.dps = 40


def conditions(w0, w1, w2, w3):
    g = [w3, w2, w1, w0, w1, w2, w3]
    e1 = sum(g) - 1
    e3 = sum(x ** 3 for x in g)
    e5 = sum(x ** 5 for x in g)
    acc, pre = mp.mpf(0), mp.mpf(0)
    for x in g:
        mid = pre + x / 2
        acc += x ** 3 * mid ** 2
        pre += x
    return [e1, e3, e5, acc]


def solve():
    return mp.findroot(lambda a, b, c, d: conditions(a, b, c, d),
                       (mp.mpf("1.3152"), mp.mpf("-1.1777"), mp.mpf("0.2356"), mp.mpf("0.7845")))


if __name__ == "__main__":
    root = solve()
    for name, v in zip(("w0", "w1", "w2", "w3"), root):
        print(name, "=", mp.nstr(v, 21))
    print("residuals:", [mp.nstr(r, 3) for r in conditions(*root)])
