"""3 -> 2 reactant rewriting ("Even for reactions involved with 3 reactants, the
reaction can also be transformed into an equivalence 2 reactants formate").

The paper gives no recipe; the one built here is the textbook one (a fast pre-equilibrium through
an intermediate complex).  A reaction of total reactant order 3 with rate constant c,

    P + Q + R -> products                      a = c * h(X),   h = prod_j C(X_j, sigma_j)

is replaced by three reactions of order <= 2 and one new species I (initial count 0):

    P + Q -> I              k_f = K * k_r      (fast)
    I     -> P + Q          k_r                (fast)
    I + R -> products       k_2 = m * c / K

with (P, Q, R) and the combinatorial factor m by the shape of the reactant row:

    A + B + C  (sigma 1,1,1):  P, Q = the two lowest species indices, R = the third;   m = 1
    2A + B     (sigma 2,1):    P = Q = A (one sigma = 2 entry),       R = B;           m = 1
    3A         (sigma 3):      P = Q = A,                             R = A;           m = 1/3

While the pair is in quasi-equilibrium, X_I ~ K * h_PQ(X), so the third reaction fires at
k_2 * X_I * X_R ~ m c h_PQ(X) X_R, which is c * h(X) in all three cases (for 3A:
C(X,2) (X-2) / 3 = C(X,3); the two molecules inside I are no longer counted in X_A).
It is an approximation, exact in the limit K -> 0 (the intermediate holds a vanishing share of
the reactant molecules: K * X_Q << 1) and k_r -> infinity (the pair equilibrates faster than
anything consumes I or changes P, Q: k_r >> k_2 * X_R).  `K` and `fast` set the two ratios:
k_r = fast * k_2 * max(1, x_scale[R]).  The price is time: the fast pair fires about 2 * fast
times per firing of the original reaction.

Host-side model transformation only: no arithmetic of the simulation method itself.
"""
import numpy as np


class RewriteError(ValueError):
    pass


def rewrite_trimolecular(net, x0, K=1e-4, fast=50.0, x_scale=None):
    """Returns (net2, x02, info): every reaction of `net` with total reactant order 3 replaced as
    described in the module docstring; all other reactions are kept, order preserved: reaction k
    of `net` becomes the block of 1 or 3 reactions starting at info["first"][k] of net2.
    info = dict(first=int64[M], origin=int64[M2] (original reaction of every new one), role=int8[M2] (0 unchanged, 1 association, 2 dissociation, 3 completion),
    intermediates=int64[n] (new species indices), n_rewritten=n)."""
    if not (K > 0.0 and fast > 0.0):
        raise RewriteError("K and fast must be positive")
    N, M = int(net["n_species"]), int(net["n_reactions"])
    rp, rs, rg = net["react_ptr"], net["react_species"], net["react_sigma"]
    sp, ss, sv = net["stoich_ptr"], net["stoich_species"], net["stoich_v"]
    rate = net["rate"]
    x0 = np.asarray(x0, dtype=np.int64)
    xs = np.maximum(1, x0 if x_scale is None else np.asarray(x_scale, dtype=np.int64))
    o_rp, o_rs, o_rg, o_sp, o_ss, o_sv, o_rate = [0], [], [], [0], [], [], []
    first, origin, role, inter = [], [], [], []

    def emit(reactants, change, c, k, what):
        for j in sorted(reactants):
            o_rs.append(j)
            o_rg.append(reactants[j])
        o_rp.append(len(o_rs))
        for j in sorted(change):
            if change[j] != 0:
                o_ss.append(j)
                o_sv.append(change[j])
        o_sp.append(len(o_ss))
        o_rate.append(c)
        origin.append(k)
        role.append(what)

    n_new = 0
    for k in range(M):
        reactants = {int(rs[e]): int(rg[e]) for e in range(rp[k], rp[k + 1])}
        change = {int(ss[e]): int(sv[e]) for e in range(sp[k], sp[k + 1])}
        order = sum(reactants.values())
        first.append(len(o_rate))
        if order <= 2:
            emit(reactants, change, float(rate[k]), k, 0)
            continue
        if order > 3:
            raise RewriteError(f"reaction {k}: total reactant order {order} > 3 is not handled")
        sig = sorted(reactants.items())                  # [(species, sigma)]
        if len(sig) == 3:
            (p, _), (q, _), (r, _) = sig
            pair, m = {p: 1, q: 1}, 1.0
        elif len(sig) == 2:
            a = sig[0][0] if sig[0][1] == 2 else sig[1][0]
            r = sig[1][0] if sig[0][1] == 2 else sig[0][0]
            pair, m = {a: 2}, 1.0
        else:
            a = r = sig[0][0]
            pair, m = {a: 2}, 1.0 / 3.0
        i_new = N + n_new
        n_new += 1
        inter.append(i_new)
        k2 = m * float(rate[k]) / K
        kr = fast * k2 * float(xs[r])
        kf = K * kr
        assoc = {j: -s for j, s in pair.items()}
        assoc[i_new] = 1
        emit(pair, assoc, kf, k, 1)
        emit({i_new: 1}, {j: -v for j, v in assoc.items()}, kr, k, 2)
        # completion: consumes I and R; the net change of the original reaction minus what the
        # association already did to P, Q
        done = dict(change)
        for j, s in pair.items():
            done[j] = done.get(j, 0) + s
        done[i_new] = -1
        emit({i_new: 1, r: 1}, done, k2, k, 3)
    net2 = dict(n_species=N + n_new, n_reactions=len(o_rate),
                react_ptr=np.asarray(o_rp, dtype=np.int64), react_species=np.asarray(o_rs, dtype=np.int32),
                react_sigma=np.asarray(o_rg, dtype=np.int32), stoich_ptr=np.asarray(o_sp, dtype=np.int64),
                stoich_species=np.asarray(o_ss, dtype=np.int32), stoich_v=np.asarray(o_sv, dtype=np.int32),
                rate=np.asarray(o_rate, dtype=np.float64))
    x02 = np.concatenate([x0, np.zeros(n_new, dtype=np.int64)])
    info = dict(first=np.asarray(first, dtype=np.int64), origin=np.asarray(origin, dtype=np.int64),
                role=np.asarray(role, dtype=np.int8), intermediates=np.asarray(inter, dtype=np.int64),
                n_rewritten=n_new)
    return net2, x02, info
