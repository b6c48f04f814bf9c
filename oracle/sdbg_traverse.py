"""oracle/sdbg_traverse.py — TEST INFRASTRUCTURE ONLY (see oracle/sdbg_oracle.c for the rules: only tests/, smoke() and
bench.py's cpu_baseline leg may use anything under oracle/; the CUDA library shares no code with it).

Traversal of the succinct de Bruijn graph, written out from the definition of the graph and not from its succinct
arrays: "A succinct de Bruijn graph (SdBG) encodes a graph with m edges in O(m) bits, and supports O(1) time traversal
from a vertex to its neighbors" (readings A24-A26 of DESIGN.md).

Input: the dict of Oracle.full_graph() — the m edges as letters ((k+1) bytes each, '$' as the outgoing symbol of a
dummy edge), sorted by (colex of the node, outgoing symbol), and the auxiliary vector of the t zero-indegree nodes.
Everything here compares node strings; nothing uses W, last or a rank/select formula. The searches below are numpy
library steps (searchsorted over reversed byte strings, one stable argsort); the definition to check by eye, in plain
loops over the same strings, is tests/helpers.py (brute_force_navigation, and boss_navigation for the formulas), and pin P13 holds this
module to it.

  node(i)      = edges[i][0..k)
  zin[i]       = 1 iff edge i is the last edge of its node and that node is one of the auxiliary vector (A24)
  F[c]         = index of the first edge whose node ends with a base >= "ACGT"[c]; F[4] = m  (the F array of Bowe et
                 al. over the last symbol of the node, in edge positions)                      (A25)
  forward(i)   = -1 for a '$' edge, else the index of the LAST edge of the node edges[i][1..k]  (A26)
  backward(j)  = the smallest i with edges[i][1..k] == node(j) and edges[i][k] != '$', or -1 when no edge enters
                 node(j)                                                                        (A26)
"""
import numpy as np


def _rev_strings(a: np.ndarray) -> np.ndarray:
    """Rows of letters -> one bytes string per row, reversed, so that bytes order is colex order (A < C < G < T)."""
    a = np.ascontiguousarray(a[:, ::-1])
    return a.view("S%d" % a.shape[1]).reshape(-1)


def navigation(full: dict, k: int) -> dict:
    E = np.asarray(full["edges"], dtype=np.uint8)
    m = E.shape[0]
    out = dict(m=m)
    if m == 0:
        out.update(zin=np.zeros(0, np.uint8), zin_bits=np.zeros(0, np.uint64), F=[0] * 5,
                   forward=np.zeros(0, np.int64), backward=np.zeros(0, np.int64))
        return out
    nodes = _rev_strings(E[:, :k])                       # non-decreasing: the edge list is sorted by colex of the node
    assert np.all(nodes[:-1] <= nodes[1:])
    last = np.ones(m, dtype=bool)
    last[:-1] = nodes[1:] != nodes[:-1]
    # A24: which edges close a node of the auxiliary vector
    aux = np.asarray(full["aux"], dtype=np.uint8).reshape(-1, k)
    auxs = _rev_strings(aux) if aux.shape[0] else np.zeros(0, dtype=nodes.dtype)
    zin = (last & np.isin(nodes, auxs)).astype(np.uint8)
    zb = np.zeros((m + 63) // 64, dtype=np.uint64)
    for i in np.nonzero(zin)[0]:                         # plain loop: the definition of the packing (LSB first)
        zb[i // 64] |= np.uint64(1) << np.uint64(i % 64)
    # A25: F over the last base of the node
    lastbase = E[:, k - 1]
    F = [int(np.searchsorted(lastbase, ord(c), side="left")) for c in "ACGT"] + [m]
    assert np.all(lastbase[:-1] <= lastbase[1:])
    # A26: forward — the last edge whose node equals edges[i][1..k]
    real = E[:, k] != ord("$")
    tgt = _rev_strings(E[:, 1:k + 1])
    fwd = np.searchsorted(nodes, tgt, side="right").astype(np.int64) - 1
    assert np.all(nodes[fwd[real]] == tgt[real])         # every target is a node (it has an edge, real or '$')
    fwd[~real] = -1
    # A26: backward — the first edge that enters node(j)
    ridx = np.nonzero(real)[0]
    order = np.argsort(tgt[ridx], kind="stable")         # equal targets keep ascending edge order
    st = tgt[ridx][order]
    pos = np.searchsorted(st, nodes, side="left")
    bwd = np.full(m, -1, dtype=np.int64)
    ok = pos < len(st)
    ok[ok] = st[pos[ok]] == nodes[ok]
    bwd[ok] = ridx[order[pos[ok]]]
    out.update(zin=zin, zin_bits=zb, F=F, forward=fwd, backward=bwd)
    return out
