"""Choice of the groups of colour flows of the helicity-shared program (gen/co_program.py) -- build-time search.

A group of colour flows shares one staging area of pair objects X (phase 2 of csrc/hs_kernel.cu); a pair object that
flows of different groups need is recomputed in each of them.  Grouping the flows by a common prefix of sigma (the
round-1 choice) recomputes 2.8 x the distinct X terms of g g -> t tbar g g g; the sharing actually follows the dihedral
orbits of sigma (rotations and reversal of the gluon word: a purely gluonic four-leg current is common to
(abcd e), (e abcd), (dcba e), (e dcba)), and a whole orbit (10 flows, 1200 staging slots) does not fit two CTAs per SM.
This module searches, deterministically (seeded simulated annealing), the partition into groups of `gsize` flows with
the smallest phase-2 cost under the staging capacity, and writes it to gen/flow_groups_n<n>.txt, which co_program reads.
PAPER.md:424-452 is the paper's version of the same trade-off (diagram groups: fewer kernels vs hand-off traffic).

  python -m paper_2510_05392_b200.gen.regroup 5        # rewrites gen/flow_groups_n5.txt (a few minutes)
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


def main(n, gsize=6, cap_slots=832, seeds=(12,), iters=1500000):
    from . import co_program
    prog = co_program.build(n, 0)
    xs = flow_xsets(prog)
    best = None
    for seed in seeds:
        r = search(xs, gsize, cap_slots, seed, iters)
        print(f"seed {seed}: cost {r[1]} max slots {r[2]}", file=sys.stderr)
        if best is None or r[1] < best[1]:
            best = r
    groups, cost, slots = best
    once = group_cost(xs, sorted(xs))[0]
    with open(path(n), "w") as f:
        f.write(f"# groups of colour flows of g g -> t tbar + {n - 2} g for the helicity-shared kernel; written by gen/regroup.py\n"
                f"# gsize {gsize}, staging capacity {cap_slots} slots: phase-2 cost {cost} (every pair object once: {once}), "
                f"largest group {slots} slots\n")
        for g in groups:
            f.write(" ".join("".join(map(str, prog.sigmas[j])) for j in g) + "\n")
    return best


if __name__ == "__main__":
    main(int(sys.argv[1]) if len(sys.argv) > 1 else 5)
