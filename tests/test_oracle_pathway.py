"""Pins of the oracle's pathway analyser (reading W1): the kinetically
fastest route between two species minimises the sum of inverse reaction rates (Dijkstra).  Pinned to a hand graph,
to the min-plus closure computed by a different algorithm (Floyd-Warshall in numpy), to the optimality conditions of
shortest paths, to the 1/c scaling, and to unreachable species."""
import numpy as np
import pytest

from conftest import SimpleNet

UNI, BI, FALLOFF, PHOTO = 0, 1, 2, 3
REV = 1 << 30


def edge_weights(net, kf, kr, n, c):
    """Dense [ns][ns] matrix of the lightest edge u -> v of column c, built from the definition with numpy
    (rates of progress from oracle-independent arithmetic: k times the product of the listed densities)."""
    ns = net.n_species
    W = np.full((ns, ns), np.inf)
    for r in range(net.n_reactions):
        for d, (frm, to, k) in enumerate(((net.reactants[r], net.products[r], kf[r, c]), (net.products[r], net.reactants[r], kr[r, c]))):
            if d == 1 and not net.reversible[r]:
                continue
            q = k * np.prod([n[s, c] for s in frm if s >= 0])
            if not (q > 0 and np.isfinite(q)):
                continue
            for u in set(int(s) for s in frm if s >= 0):
                for v in set(int(s) for s in to if s >= 0):
                    if u != v:
                        W[u, v] = min(W[u, v], 1.0 / q)
    return W


def floyd_warshall(W):
    D = W.copy()
    np.fill_diagonal(D, 0.0)
    for k in range(D.shape[0]):
        D = np.minimum(D, D[:, k:k + 1] + D[k:k + 1, :])
    return D


def test_two_step_route_beats_the_direct_one_exactly_when_it_is_faster(oracle):
    """X0 -> X1 (rate q1), X1 -> X2 (q2), X0 -> X2 (q3): the route through X1 costs 1/q1 + 1/q2."""
    z = np.zeros((3, 7))
    net = SimpleNet(np.ones((3, 1)), z, z, [1000.0] * 3, [UNI, UNI, UNI], [[0], [1], [0]], [[1], [2], [2]], [0, 0, 0], np.zeros((3, 3)))
    n = np.array([[2.0, 2.0], [4.0, 4.0], [1.0, 1.0]])
    kf = np.array([[5.0, 5.0], [2.0, 2.0], [1.0, 0.2]])                      # q = (10, 8, 2) and (10, 8, 0.4)
    dist, pred, via = oracle.pathway(net, kf, np.zeros_like(kf), n, 0)
    assert np.allclose(dist[:, 0], [0.0, 0.1, 0.225]) and np.allclose(dist[:, 1], [0.0, 0.1, 0.225])   # 1/10 + 1/8 = 0.225 < 1/2, 1/0.4
    assert pred[2, 0] == 1 and via[2, 0] == 1 and pred[1, 0] == 0 and via[1, 0] == 0 and pred[0, 0] == -1
    kf[2] = [20.0, 4.0]                                                      # q3 = 40: direct (0.025); q3 = 8: direct 0.125 < 0.225
    dist, pred, via = oracle.pathway(net, kf, np.zeros_like(kf), n, 0)
    assert np.allclose(dist[2], [0.025, 0.125]) and np.all(pred[2] == 0) and np.all(via[2] == 2)
    # X2 cannot reach anything (no reverse): unreachable species are +inf with pred = via = -1
    dist, pred, via = oracle.pathway(net, kf, np.zeros_like(kf), n, 2)
    assert dist[2, 0] == 0.0 and np.all(np.isinf(dist[:2])) and np.all(pred == -1) and np.all(via == -1)


def test_reverse_directions_and_multi_species_reactions_form_edges(oracle):
    """X0 + X1 <=> X2 + X3: forward edges X0->X2, X0->X3, X1->X2, X1->X3 of weight 1/q_f, reverse edges the other way
    of weight 1/q_r; the via word carries the direction bit."""
    z = np.zeros((4, 7))
    net = SimpleNet(np.ones((4, 1)), z, z, [1000.0] * 4, [BI], [[0, 1]], [[2, 3]], [1], np.zeros((1, 3)))
    n = np.array([[2.0], [3.0], [5.0], [7.0]])
    kf, kr = np.array([[0.5]]), np.array([[0.1]])                              # q_f = 3, q_r = 3.5
    dist, pred, via = oracle.pathway(net, kf, kr, n, 0)
    assert np.allclose(dist[:, 0], [0.0, 1 / 3 + 1 / 3.5, 1 / 3, 1 / 3])
    assert via[2, 0] == 0 and via[1, 0] == (0 | REV) and pred[1, 0] in (2, 3)


@pytest.mark.parametrize("cfg", [1, 2])
def test_distances_equal_the_min_plus_closure_and_satisfy_the_optimality_conditions(oracle, network, cfg):
    from paper_2512_06729_b200 import synth
    net = network(cfg)
    atm = synth.config_atmosphere(cfg, net)
    ncol = 3
    kf, kr = oracle.rate_coeffs(net, atm.T, atm.P, atm.J, ncol)
    n = atm.n
    for c in range(ncol):
        W = edge_weights(net, kf, kr, n, c)
        closure = floyd_warshall(W)
        for source in (0, net.n_species // 2, net.n_species - 1):
            dist, pred, via = oracle.pathway(net, kf, kr, n, source, ncol)
            d = dist[:, c]
            fin = np.isfinite(closure[source])
            assert np.array_equal(np.isfinite(d), fin)
            assert np.allclose(d[fin], closure[source][fin], rtol=1e-13, atol=0)
            # optimality: no edge can shorten any distance; every tree edge is tight
            with np.errstate(invalid="ignore"):
                slack = d[:, None] + W - d[None, :]
            ok = np.isfinite(slack)
            assert np.all(slack[ok] >= -1e-13 * np.broadcast_to(d[None, :], slack.shape)[ok])
            for v in range(net.n_species):
                if v == source or not np.isfinite(d[v]):
                    assert pred[v, c] == -1 and via[v, c] == -1
                    continue
                u, r, rev = pred[v, c], via[v, c] & ~REV, bool(via[v, c] & REV)
                frm, to = (net.products[r], net.reactants[r]) if rev else (net.reactants[r], net.products[r])
                assert u in frm and v in to
                k = (kr if rev else kf)[r, c]
                w = 1.0 / (k * np.prod([n[s, c] for s in frm if s >= 0]))
                assert abs(d[u] + w - d[v]) <= 1e-13 * d[v]


def test_distances_scale_inversely_with_all_rates(oracle, network):
    from paper_2512_06729_b200 import synth
    net = network(1)
    atm = synth.config_atmosphere(1, net)
    kf, kr = oracle.rate_coeffs(net, atm.T, atm.P, atm.J, 4)
    d1, _, _ = oracle.pathway(net, kf, kr, atm.n, 3, 4)
    d2, _, _ = oracle.pathway(net, 8.0 * kf, 8.0 * kr, atm.n, 3, 4)
    fin = np.isfinite(d1[:, :4])
    assert np.array_equal(np.isfinite(d2[:, :4]), fin)
    assert np.array_equal(d2[:, :4][fin] * 8.0, d1[:, :4][fin])              # a power of two: exact
