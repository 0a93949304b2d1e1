"""Host-side generator (diagram enumeration, colour algebra, lowering to the diagram program) on CPU.

Pins: Table 2 of the paper (tests/golden/table2_complexity.txt), the oracle's brute-force colour matrix,
and the oracle's per-helicity matrix elements through the numpy IR evaluator tests/ir_eval.py.
"""
import math
import os

import numpy as np
import pytest

import ir_eval
import oracle
from paper_2510_05392_b200 import inputs
from paper_2510_05392_b200.gen import colour, diagrams

HERE = os.path.dirname(os.path.abspath(__file__))


def _table2():
    rows = {}
    for line in open(os.path.join(HERE, "golden", "table2_complexity.txt")):
        if line.startswith("#") or not line.strip():
            continue
        name, nd, nc, nh, nw = line.split()
        rows[name] = (int(nd), int(nc), int(nh), int(nw))
    return rows


@pytest.mark.parametrize("n", [2, 3, 4, 5])
def test_diagram_and_colour_counts_match_table2(n):
    t2 = _table2()
    proc = diagrams.build_process(n)
    nd, nc, nh, _ = t2[proc.name]
    assert proc.ndiagrams == nd
    assert proc.ncolor == nc == math.factorial(n)
    assert 2 ** proc.npar == nh
    # every diagram appears in the program, four-gluon vertices as three terms each
    assert len({a.diagram for a in proc.amps}) == nd


def test_diagram_count_recursion_p7():
    """psi(n) = sum_j C(n,j) g(j) psi(n-j) with g = 1,1,4,25,220,2485 reproduces Table 2 up to 2->6."""
    g = [len(diagrams.gluon_trees(tuple(range(k)))) for k in range(1, 7)]
    assert g == [1, 1, 4, 25, 220, 2485]
    psi = [1]
    for n in range(1, 7):
        psi.append(sum(math.comb(n, j) * g[j - 1] * psi[n - j] for j in range(1, n + 1)))
    t2 = _table2()
    assert psi[2:7] == [t2[k][0] for k in ("gg_ttx", "gg_ttxg", "gg_ttxgg", "gg_ttxggg", "gg_ttxgggg")]


@pytest.mark.parametrize("n", [2, 3, 4, 5])
def test_exact_colour_matrix_matches_oracle_brute_force(n):
    C = colour.colour_matrix(n)
    den = colour.common_denominator(C)
    assert den == {2: 3, 3: 9, 4: 54, 5: 324}[n]
    Cf = np.array([[float(x) for x in r] for r in C])
    np.testing.assert_allclose(Cf, oracle.color_matrix(n), atol=1e-11)
    ints = np.array([[int(x * den) for x in r] for r in C])
    assert np.abs(ints).max() <= 4096          # exactly representable in TF32 (11-bit significand incl. hidden bit)


@pytest.mark.parametrize("name,n,hels", [("gg_ttx", 2, None), ("gg_ttxg", 3, None), ("gg_ttxgg", 4, None),
                                         ("gg_ttxggg", 5, (0, 37, 100, 127))])
def test_program_matches_oracle_per_helicity(name, n, hels, params):
    proc = diagrams.build_process(n)
    C = np.array([[float(x) for x in r] for r in colour.colour_matrix(n)])
    gs = math.sqrt(4 * math.pi * params["aS"])
    p = inputs.momenta(name, 2, seed=3)
    _, mh_o = oracle.matrix_elements(name, p, params, per_helicity=True)
    npar = proc.npar
    for h in (range(1 << npar) if hels is None else hels):
        hel = [1 if (h >> (npar - 1 - i)) & 1 else -1 for i in range(npar)]
        j = ir_eval.evaluate(proc, p[1], hel, params["mT"], params["wT"])
        mh = (j.conj() @ C @ j).real * gs ** (2 * n) / oracle.DENOM[name]
        assert abs(mh / mh_o[1][h] - 1) < 1e-10, (h, mh, mh_o[1][h])


@pytest.mark.parametrize("name,n,nev", [("gg_ttxgg", 4, 2), ("gg_ttxggg", 5, 1)])
def test_helicity_shared_streams_match_oracle(name, n, nev, params):
    """the device streams of the helicity-shared kernel (gen/hs_streams.py: merged four-gluon vertices, X.Y split, chunks,
    classes, packed offsets), interpreted lane by lane by tests/hs_eval.py, give the oracle's per-helicity colour-summed
    |M|^2 for EVERY helicity -- the program that is the default for these processes, checked without a GPU"""
    import hs_eval
    from paper_2510_05392_b200.gen import emit_hs, hs_streams
    k = emit_hs.KERNEL_CFG[n]
    st = emit_hs.streams(n)                                                        # what the library is built with
    T = st.tables()
    # the static schedule deals every colour flow and every chunk of every step to exactly one warp, units unbroken
    for s_, (g3, g2) in enumerate(st.steps()):
        want_f = list(range(int(T["grp"][g3][2]), int(T["grp"][g3][2] + T["grp"][g3][3]))) if g3 is not None else []
        want_c = []
        if g2 is not None:
            u0, nu = int(T["grp"][g2][0]), int(T["grp"][g2][1])
            for u in range(u0, u0 + nu):
                want_c += list(range(int(T["p2unit"][u][0]), int(T["p2unit"][u][0] + T["p2unit"][u][1])))
        got_f, got_c = [], []
        for w in range(k["nw"]):
            sf, sc = (int(x) for x in T["wsched"][s_ * k["nw"] + w])
            got_f += [int(x) for x in T["witem"][sf & 0xFFFF:(sf & 0xFFFF) + (sf >> 16)]]
            run = list(range(sc & 0xFFFF, (sc & 0xFFFF) + (sc >> 16)))
            got_c += run
            if run:          # a run starts with the first chunk of a unit and ends with the last chunk of one
                assert (int(T["p2rec"][run[0]][0, 0, 1]) >> 12) & 1 and (int(T["p2rec"][run[-1]][0, 0, 1]) >> 13) & 1
        assert sorted(got_f) == want_f and sorted(got_c) == sorted(want_c), s_
    C = np.array([[float(x) for x in r] for r in colour.colour_matrix(n)])
    gs = math.sqrt(4 * math.pi * params["aS"])
    p = inputs.momenta(name, nev, seed=7)
    _, mh_o = oracle.matrix_elements(name, p, params, per_helicity=True)
    for e in range(nev):
        J = hs_eval.evaluate(T, p[e], params["mT"], params["wT"])
        mh = np.einsum("ih,ij,jh->h", J.conj(), C, J).real * gs ** (2 * n) / oracle.DENOM[name]
        assert np.abs(mh / mh_o[e] - 1).max() < 1e-10


@pytest.mark.parametrize("name,n", [("gg_ttxgg", 4), ("gg_ttxggg", 5), ("gg_ttxgggg", 6)])
def test_generic_tables_match_oracle(name, n, params):
    """the tables of the generic helicity-shared kernel (gen/hsg_tables.py; the program of g g -> t tbar g g g g with its
    4-leg colour-ordered objects, Table 2 at PAPER.md:180-187), interpreted by tests/hsg_eval.py, give the oracle's
    per-helicity colour-summed |M|^2 for EVERY helicity (colour matrix: the oracle's, brute force)"""
    import hsg_eval
    from paper_2510_05392_b200.gen import hsg_tables
    T = hsg_tables.tables(n)
    assert T["ncolor"] == math.factorial(n) and len(T["flow"]) == T["ncolor"]
    C = oracle.color_matrix(n)
    gs = math.sqrt(4 * math.pi * params["aS"])
    p = inputs.momenta(name, 1, seed=7)
    _, mh_o = oracle.matrix_elements(name, p, params, per_helicity=True)
    J = hsg_eval.evaluate(T, p[0], params["mT"], params["wT"])
    mh = np.einsum("ih,ij,jh->h", J.conj(), C, J).real * gs ** (2 * n) / oracle.DENOM[name]
    assert np.abs(mh / mh_o[0] - 1).max() < 1e-9
    if n == 6:
        # the tables of phase 3 on the FP64 tensor path (classes, fragment offsets, staged layout, swizzled accumulator),
        # executed lane by lane as the kernel does, give the same jamps: every 24th colour flow, all 256 helicities
        fl = set(range(0, len(T["flow"]), 24))
        Jt = hsg_eval.evaluate_tensor(T, p[0], params["mT"], params["wT"], flows=fl)
        assert set(int(x) for x in T["flow"][:, 3]) <= {3, 4}                  # classes per flow
        for f in fl:
            j = int(T["flow"][f][0])
            assert np.abs(Jt[j] - J[j]).max() < 1e-12 * np.abs(J[j]).max()
