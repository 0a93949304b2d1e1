"""Choice of the groups of colour flows of the helicity-shared program (gen/co_program.py) -- build-time search.

A group of colour flows shares one staging area of pair objects X (phase 2 of csrc/hs_kernel.cu); a pair object that
flows of different groups need is recomputed in each of them.  Grouping the flows by a common prefix of sigma (the
round-1 choice) recomputes 2.8 x the distinct X terms of g g -> t tbar g g g; the sharing actually follows the dihedral
orbits of sigma (rotations and reversal of the gluon word: a purely gluonic four-leg current is common to
(abcd e), (e abcd), (dcba e), (e dcba)).  One orbit = 10 flows and 1200 staging slots (77 KB); the kernel therefore runs
one 16-warp CTA per SM with a double-buffered staging area.  `main` writes the orbit partition to
gen/flow_groups_n<n>.txt, which co_program reads; `search` (seeded simulated annealing under a staging capacity) is the
generic tool for other group sizes (6 flows within 832 slots: cost 4.65e6 against 4.20e6 for the orbits and 6.67e6 for
prefix groups).  PAPER.md:424-452 is the paper's version of the same trade-off (diagram groups: fewer kernels against
hand-off traffic).

  python -m paper_2510_05392_b200.gen.regroup 5        # rewrites gen/flow_groups_n5.txt
"""
from __future__ import annotations

import math
import os
import random
import sys

HERE = os.path.dirname(os.path.abspath(__file__))

# relative cost of a phase-2 term (flops of emit_hs.FLOPS + accumulation)
X_COST = {"x_row": 72, "x_col": 72, "x_bil": 80, "x_v3": 134, "x_v4": 112, "x_v4s": 170}


def path(n):
    return os.path.join(HERE, f"flow_groups_n{n}.txt")


def flow_xsets(prog):
    """per colour flow j: {pair-object key: (staging slots, phase-2 cost)} from the single-group program"""
    assert len(prog.groups) == 1
    g = prog.groups[0]
    out = {}
    for j, ents in g["entries"].items():
        d = {}
        for xs, _, _ in ents:
            x = g["xobjs"][xs]
            nv = 1 << len(x["legs"])
            d[xs] = (nv, nv * sum(X_COST[t.op] for t in x["terms"]))
        out[j] = d
    return out


def group_cost(xsets, members):
    seen = {}
    for j in members:
        seen.update(xsets[j])
    return sum(c for _, c in seen.values()), sum(s for s, _ in seen.values())


def search(xsets, gsize, cap_slots, seed=0, iters=600000):
    """partition of the flows into groups of `gsize` minimising the summed phase-2 cost, every group within `cap_slots`"""
    rnd = random.Random(seed)
    flows = sorted(xsets)
    assert len(flows) % gsize == 0
    order = flows[:]
    rnd.shuffle(order)
    ng = len(flows) // gsize
    groups = [order[i * gsize:(i + 1) * gsize] for i in range(ng)]
    pen = lambda cs: cs[0] + 3000 * max(0, cs[1] - cap_slots)
    gc = [group_cost(xsets, g) for g in groups]
    temp = 20000.0
    for _ in range(iters):
        a, b = rnd.sample(range(ng), 2)
        i, j = rnd.randrange(gsize), rnd.randrange(gsize)
        ga, gb = groups[a][:], groups[b][:]
        ga[i], gb[j] = gb[j], ga[i]
        ca, cb = group_cost(xsets, ga), group_cost(xsets, gb)
        d = pen(ca) + pen(cb) - pen(gc[a]) - pen(gc[b])
        if d <= 0 or rnd.random() < math.exp(-d / temp):
            groups[a], groups[b], gc[a], gc[b] = ga, gb, ca, cb
        temp = max(50.0, temp * 0.99999)
    assert all(s <= cap_slots for _, s in gc), "no partition within the staging capacity found"
    groups = sorted(sorted(g) for g in groups)
    return groups, sum(c for c, _ in gc), max(s for _, s in gc)


def load(n, sigmas):
    """groups of flow indices from gen/flow_groups_n<n>.txt (one group per line, flows as gluon words)"""
    index = {"".join(map(str, s)): j for j, s in enumerate(sigmas)}
    groups = []
    for line in open(path(n)):
        line = line.split("#")[0].split()
        if line:
            groups.append([index[w] for w in line])
    assert sorted(j for g in groups for j in g) == list(range(len(sigmas))), "flow_groups file is not a partition"
    return groups


def dihedral_orbits(sigmas):
    """orbits of the colour flows under rotations and reversal of the gluon word"""
    index = {tuple(s): j for j, s in enumerate(sigmas)}
    seen, out = set(), []
    for j, s_ in enumerate(sigmas):
        if j in seen:
            continue
        s_ = tuple(s_)
        orb = set()
        for r in range(len(s_)):
            t = s_[r:] + s_[:r]
            orb |= {index[t], index[t[::-1]]}
        seen |= orb
        out.append(sorted(orb))
    return out


def main(n):
    from . import co_program
    prog = co_program.build(n, 0)
    xs = flow_xsets(prog)
    groups = dihedral_orbits(prog.sigmas)
    costs = [group_cost(xs, g) for g in groups]
    cost, slots = sum(c for c, _ in costs), max(s_ for _, s_ in costs)
    once = group_cost(xs, sorted(xs))[0]
    with open(path(n), "w") as f:
        f.write(f"# groups of colour flows of g g -> t tbar + {n - 2} g for the helicity-shared kernel; written by gen/regroup.py\n"
                f"# dihedral orbits of the gluon word: phase-2 cost {cost} (every pair object once: {once}), "
                f"largest group {slots} staging slots\n")
        for g in groups:
            f.write(" ".join("".join(map(str, prog.sigmas[j])) for j in g) + "\n")
    return groups, cost, slots


if __name__ == "__main__":
    main(int(sys.argv[1]) if len(sys.argv) > 1 else 5)
