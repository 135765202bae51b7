"""Networks and checkpointed states whose waiting times tie EXACTLY (reading G6 of DESIGN.md:
PAPER.md:162-164, Eq.25 "first arriving wins all" is silent on ties; lowest index wins).

Input construction only -- no arithmetic of the method.  Every number below is chosen so that the
products and quotients the method forms are exact in binary64 (powers of two times a double), so
the expected outcome follows by hand, independent of any implementation:

  * every channel k starts with T_k = 0, P_k = 8 * a_k(X0)        (an exact scaling)
    -> dt_k = P_k / a_k = 8.0 for EVERY k: an M-way finite tie at dt = 8; channel 0 fires at t = 8;
  * then T_k = a_k * 8 = P_k exactly, residual 0 for every channel that has not fired yet, and
    0 / a = 0 whatever the refreshed a_k > 0 is: an (M-1)-way tie at dt = 0; channel 1 fires; ...
  * a fired channel's target moves by a fresh exponential (> 0), so it is out of the race.

Expected trace: mu = 0, 1, 2, ..., M-1, every event at t = 8.0 exactly.
"""
import numpy as np

import rt_workloads as W

H0 = 4           # initial count of the hub species (a power of two: c_k * H0 is exact)


def tie_network(M, n_species=8, seed=0, coupled=True):
    """M channels.  coupled=False: pure sources 0 -> S_j (no reactants, nothing is ever refreshed).
    coupled=True: a mix of sources, hub readers H -> 2H + S_j (every firing of one changes H, so
    EVERY reader is refreshed every firing: the dependency walk, staging rounds and the "refreshed
    reaction joins the reduction as a fresh candidate" path all run inside the tie) and catalysed
    hub readers H + S_1 -> 2H + S_1 + S_j (two reactants; S_1 = 2 stays constant, S_1 is only
    ever produced by nobody).  Returns (net, x0, T0, P0, n0)."""
    rng = np.random.default_rng(seed)
    c = rng.uniform(0.5, 2.0, size=M)
    reactions, a0 = [], np.empty(M)
    for k in range(M):
        j = 2 + k % (n_species - 2)
        kind = (k % 3) if coupled else 0
        if kind == 0:
            reactions.append(({}, {j: 1}, float(c[k])))
            a0[k] = c[k]
        elif kind == 1:
            reactions.append(({0: 1}, {0: 2, j: 1}, float(c[k])))
            a0[k] = c[k] * H0                 # exact
        else:
            reactions.append(({0: 1, 1: 1}, {0: 2, 1: 1, j: 1}, float(c[k])))
            a0[k] = c[k] * H0 * 2             # exact (S_1 = 2)
    net = W.from_reactions(n_species, reactions)
    x0 = np.zeros(n_species, dtype=np.int64)
    x0[0], x0[1] = H0, 2
    T0 = np.zeros(M)
    P0 = a0 * 8.0                              # exact
    n0 = np.zeros(M, dtype=np.uint64)
    return net, x0, T0, P0, n0


def expected_trace(M):
    return np.arange(M, dtype=np.int32), np.full(M, 8.0)
