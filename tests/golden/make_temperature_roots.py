"""Writes tests/golden/temperature_roots.txt: closed-form optimal temperatures T* of Problem 1 for
geometric logits z_i = -lam * i under the SNAPKV max-pool metric of radius r (L278), used to pin Algorithm 2 (L625-648).

Derivation (no oracle code involved; scipy only).  rho = e^-lam.  The raw scores S_i ~ rho^i give the Top-p count
k = ceil(ln(1 - p (1 - rho^N)) / ln rho) (pin P5) and M_k(S) = (1 - rho^k) / (1 - rho^N).  Max-pooling with radius r maps
z_i to z_{max(i - r, 0)}: r + 1 copies of the top logit followed by the same geometric tail, so with q = e^{-lam / T}
M_k(S_hat(T)) = (r + geo(k - r)) / (r + geo(N - r)),  geo(m) = (1 - q^m) / (1 - q)   (k > r).
T* solves M_k(S) = M_k(S_hat(T)); brentq on [0.25, 4].

Run:  python tests/golden/make_temperature_roots.py
"""
import math
import os

import scipy.optimize

CASES = [(0.1, 400, 5, 0.9), (0.05, 800, 3, 0.9), (0.1, 400, 5, 0.95), (0.2, 300, 2, 0.8), (0.02, 1500, 7, 0.9)]


def root(lam, N, r, p):
    rho = math.exp(-lam)
    k = math.ceil(math.log(1 - p * (1 - rho ** N)) / math.log(rho))
    assert k > r
    mks = (1 - rho ** k) / (1 - rho ** N)

    def f(T):
        q = math.exp(-lam / T)
        geo = lambda m: (1 - q ** m) / (1 - q)
        return mks - (r + geo(k - r)) / (r + geo(N - r))

    return k, scipy.optimize.brentq(f, 0.25, 4.0, xtol=1e-12)


if __name__ == "__main__":
    out = os.path.join(os.path.dirname(os.path.abspath(__file__)), "temperature_roots.txt")
    with open(out, "w") as fh:
        fh.write("# lam N r p k T_star  -- closed-form roots of Problem 1 (PAPER.md L108-110) for z_i = -lam*i under a\n"
                 "# max-pool of radius r (L278); derivation and generator: make_temperature_roots.py (scipy only)\n")
        for lam, N, r, p in CASES:
            k, T = root(lam, N, r, p)
            fh.write(f"{lam} {N} {r} {p} {k} {T:.9f}\n")
    print(open(out).read())
