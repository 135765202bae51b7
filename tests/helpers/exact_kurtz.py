"""Exact (rational-arithmetic) sample path of the random time-change representation
    X(t) = X(0) + sum_k Y_k(T_k(t)) v_k,   T_k(t) = int_0^t a_k(X(s)) ds      (Eq.15-16)
for GIVEN jump times of the unit-rate Poisson processes Y_k.

The jump times are inputs (partial sums of the exponential increments E(k,0), E(k,1), ...);
everything else is python Fractions and math.comb, so there is no rounding and no shared code
with the oracle.  Between two firings every a_k is constant, T_k is linear in t, and channel k
reaches its next jump time J_k after (J_k - T_k)/a_k of real time; the earliest one fires
(Eq.24-25).  Brute force: O(M) exact work per firing, tiny networks only.
"""
from fractions import Fraction
from math import comb


def exact_path(net, x0, draw, n_firings):
    """draw(k, n) -> float increment E(k,n).  Returns list of (mu, t as Fraction) and final X."""
    M = int(net["n_reactions"])
    rp, rs, rg = net["react_ptr"], net["react_species"], net["react_sigma"]
    sp, ss, sv = net["stoich_ptr"], net["stoich_species"], net["stoich_v"]
    X = [int(v) for v in x0]
    T = [Fraction(0)] * M
    n = [0] * M
    J = [Fraction(draw(k, 0)) for k in range(M)]
    t = Fraction(0)
    path = []
    for _ in range(n_firings):
        a = []
        for k in range(M):
            h = 1
            for e in range(rp[k], rp[k + 1]):
                h *= comb(X[rs[e]], int(rg[e]))
            a.append(Fraction(float(net["rate"][k])) * h)
        best, mu = None, -1
        for k in range(M):
            if a[k] > 0:
                w = (J[k] - T[k]) / a[k]
                if best is None or w < best:
                    best, mu = w, k
        if best is None:
            break
        t += best
        for k in range(M):
            T[k] += a[k] * best
        for e in range(sp[mu], sp[mu + 1]):
            X[ss[e]] += int(sv[e])
        n[mu] += 1
        J[mu] += Fraction(draw(mu, n[mu]))
        path.append((mu, t))
    return path, X
