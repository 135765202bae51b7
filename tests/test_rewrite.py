"""3 -> 2 reactant rewriting: structure of the rewritten network, agreement in
distribution with the original sigma = 3 network on small cases (oracle on both sides, so this
checks the transformation, not the CUDA path), and one run of a rewritten network on the GPU."""
import math

import numpy as np
import pytest
from scipy import stats

import rt_workloads as W
from paper_2103_00405_b200.rewrite import RewriteError, rewrite_trimolecular


def _orders(net):
    rp, rg = net["react_ptr"], net["react_sigma"]
    return [int(rg[rp[k]:rp[k + 1]].sum()) for k in range(net["n_reactions"])]


def _mixed_network():
    # 0: A+B+C -> D   1: 2A+B -> D+A   2: 3A -> B   3: A -> 0 (kept)   4: B+C -> A (kept)   5: A+2C -> D
    reactions = [({0: 1, 1: 1, 2: 1}, {3: 1}, 2e-4), ({0: 2, 1: 1}, {3: 1, 0: 1}, 3e-4),
                 ({0: 3}, {1: 1}, 1e-4), ({0: 1}, {}, 0.05), ({1: 1, 2: 1}, {0: 1}, 1e-3),
                 ({0: 1, 2: 2}, {3: 1}, 2e-4)]
    return W.from_reactions(4, reactions), np.array([30, 25, 35, 0], dtype=np.int64)


def test_structure_of_the_rewritten_network():
    import paper_2103_00405_b200 as rt
    net, x0 = _mixed_network()
    assert max(_orders(net)) == 3
    net2, x02, info = rewrite_trimolecular(net, x0, K=1e-3, fast=20.0)
    assert info["n_rewritten"] == 4 and net2["n_species"] == 8 and net2["n_reactions"] == 2 + 4 * 3
    assert max(_orders(net2)) == 2                                   # <= 2 reactant molecules per row
    assert list(info["first"]) == [0, 3, 6, 9, 10, 11]
    assert list(info["role"]) == [1, 2, 3, 1, 2, 3, 1, 2, 3, 0, 0, 1, 2, 3]
    assert list(x02) == [30, 25, 35, 0, 0, 0, 0, 0]
    assert rt.rt_validate_network(net2) == rt.RT_OK                  # (host-side check of the C ABI)
    sp, ss, sv = net2["stoich_ptr"], net2["stoich_species"], net2["stoich_v"]
    rows = [dict(zip(ss[sp[k]:sp[k + 1]].tolist(), sv[sp[k]:sp[k + 1]].tolist())) for k in range(14)]
    # association + completion together make the original net change (intermediate cancels)
    osp, oss, osv = net["stoich_ptr"], net["stoich_species"], net["stoich_v"]
    for k in (0, 1, 2, 5):
        f = int(info["first"][k])
        total = {}
        for row in (rows[f], rows[f + 2]):
            for j, v in row.items():
                total[j] = total.get(j, 0) + v
        total = {j: v for j, v in total.items() if v != 0}
        assert total == dict(zip(oss[osp[k]:osp[k + 1]].tolist(), osv[osp[k]:osp[k + 1]].tolist())), k
        assert rows[f + 1] == {j: -v for j, v in rows[f].items()}    # dissociation undoes association
    # rates: k_f / k_r = K, k_2 = m c / K with m = 1/3 for 3A
    r = net2["rate"]
    assert r[0] / r[1] == pytest.approx(1e-3) and r[2] == pytest.approx(2e-4 / 1e-3)
    assert r[8] == pytest.approx(1e-4 / 3 / 1e-3) and r[7] == pytest.approx(20.0 * r[8] * 30)
    with pytest.raises(RewriteError):
        rewrite_trimolecular(W.from_reactions(2, [({0: 2, 1: 2}, {1: 1}, 1.0)]), [5, 5])


@pytest.mark.parametrize("which", ["A+B+C", "2A+B", "3A"])
def test_rewritten_network_agrees_in_distribution(which):
    """Oracle on the sigma = 3 network vs oracle on the rewritten one (different seeds): product
    count at t_end, two-sample KS p > 0.01 and means within 3 SE."""
    import oracle
    if which == "A+B+C":
        net, x0 = W.from_reactions(4, [({0: 1, 1: 1, 2: 1}, {3: 1}, 4e-4)]), [30, 40, 35, 0]
    elif which == "2A+B":
        net, x0 = W.from_reactions(3, [({0: 2, 1: 1}, {2: 1}, 6e-4)]), [40, 30, 0]
    else:
        net, x0 = W.from_reactions(2, [({0: 3}, {1: 1}, 6e-4)]), [45, 0]
    x0 = np.asarray(x0, dtype=np.int64)
    prod = len(x0) - 1
    net2, x02, info = rewrite_trimolecular(net, x0, K=2e-5, fast=40.0)
    n, t_end = 400, 1.0
    a = oracle.ensemble(net, x0, 3, 0, n, 0, t_end, n_threads=8)["x"][:, prod].astype(float)
    r2 = oracle.ensemble(net2, x02, 4, 0, n, 0, t_end, n_threads=8)
    b = r2["x"][:, prod].astype(float)
    assert 3 < a.mean() < x0[0] / (3 if which == "3A" else 1) - 3     # (a non-trivial regime)
    assert stats.ks_2samp(a, b).pvalue > 0.01
    se = math.sqrt(a.var(ddof=1) / n + b.var(ddof=1) / n)
    assert abs(a.mean() - b.mean()) < 3 * se
    assert r2["x"][:, info["intermediates"][0]].mean() < 0.2          # the complex stays rare


@pytest.mark.gpu
def test_rewritten_network_runs_on_the_gpu_bit_exact():
    import oracle
    import paper_2103_00405_b200 as rt
    net, x0 = _mixed_network()
    net2, x02, info = rewrite_trimolecular(net, x0, K=1e-3, fast=20.0)
    o = oracle.run(net2, x02, 9, 0, 3000, math.inf, 3000)
    with rt.Model(net2) as m:
        g = m.run(x02, 9, 0, 3000, math.inf, 3000)
        ens = m.ensemble(x02, 9, 0, 5, 2000, math.inf)
    np.testing.assert_array_equal(g["trace_mu"], o["trace_mu"])
    np.testing.assert_array_equal(g["x"], o["x"])
    np.testing.assert_allclose(g["trace_t"], o["trace_t"], rtol=1e-12, atol=0)
    oe = oracle.ensemble(net2, x02, 9, 0, 5, 2000, math.inf)
    np.testing.assert_array_equal(ens["x"], oe["x"])
