"""numpy interpreter of the device streams of the helicity-shared program (gen/hs_streams.py) -- CPU TEST HELPER.

Executes, lane by lane, exactly what one CTA of csrc/hs_kernel.cu executes for one event: the same packed records, the
same byte offsets into the shared-memory planes, the same fragment <-> (row, column, tile) conventions of the FP64
tensor-core tiles and the same accumulator slots -- but every opcode is restated with the plain gamma-matrix helpers of
tests/ir_eval.py.  So the generator's factorisation (merge_v4_pairs, the X.Y split and its signs, chunking, classes,
packing) is checked against the oracle on CPU before any kernel runs.  Not product, not oracle; nothing here is imported
by the package.
"""
import numpy as np

import ir_eval as ir

G = ir.G


def _perm(v):
    return (v & ~1) | (bin(v).count("1") & 1)


def _sub(v, code):
    return sum(((v >> ((code >> (3 * j)) & 7)) & 1) << j for j in range(3))


def _acc_swizzle(h):
    hi = h >> 3
    return h ^ (((hi & 1) * 3) ^ (((hi >> 1) & 1) * 5) ^ (((hi >> 2) & 1) * 6) ^ (((hi >> 3) & 1) * 7))


class _Planes:
    """an area of four component planes; addressed by the byte offset inside plane 0 like the kernel does"""

    def __init__(self, plane_bytes):
        assert plane_bytes % 128 == 32
        self.a = np.full((4, plane_bytes // 16), np.nan + 0j, dtype=complex)

    def load(self, off):
        assert off % 16 == 0
        return self.a[:, off // 16].copy()

    def store(self, off, val):
        self.a[:, off // 16] = val


def _x_term(op, A, B, Z, kA, kB):
    if op == 8:
        return A @ ir.slash(B)
    if op == 9:
        return ir.slash(A) @ B
    if op == 10:
        return G * np.array([A @ ir.GAM[mu] @ B for mu in range(4)])
    if op == 11:
        return G * (ir.mdot(A, B) * (kA - kB) + ir.mdot(2 * kB + kA, A) * B - ir.mdot(2 * kA + kB, B) * A)
    if op == 12:
        return G * (ir.mdot(A, Z) * B - ir.mdot(B, Z) * A)
    if op == 13:
        return G * (2 * ir.mdot(A, Z) * B - ir.mdot(B, Z) * A - ir.mdot(A, B) * Z)
    raise ValueError(op)


def evaluate(T, mom, mt, wt):
    """jamps[ncolor][2^npar] (without the g^n factor) of one event from the streams T = Streams.tables()"""
    npar, ntile = T["npar"], T["ntile"]
    k = [mom[i] * (1 if i < 2 else -1) for i in range(npar)]
    K = [sum(k[p] for p in range(npar) if (m >> p) & 1) for m in T["legset_mask"]]
    obj = _Planes(T["obj_plane"])

    # phase 1: colour-ordered objects, level by level (term table interpreted directly)
    def arg(w, var):
        return obj.load(16 * ((w & 0xFFFF) + _perm(_sub(var, (w >> 16) & 0x1FF))))

    for it in T["p1_items"]:
        if int(it) < 0:                       # idle lane of a block
            continue
        o, var = int(it) >> 8, int(it) & 0xFF
        slot0, info, t0, nt = (int(x) for x in T["obj"][o])
        kout = K[info >> 8]
        acc = np.zeros(4, dtype=complex)
        for t in T["term"][t0:t0 + nt]:
            w0, w1, w2, w3 = (int(x) & 0xFFFFFFFF for x in t)
            op, neg = w0 & 0xFF, (w0 >> 8) & 1
            hel = 1 if var & 1 else -1
            if op == 0:
                e = ir.polvec(mom[w1], hel)
                r = e if w1 < 2 else e.conj()
            elif op == 1:
                r = ir.u_spinor(mom[2], mt, hel).conj() @ ir.GAM[0]
            elif op == 2:
                r = ir.v_spinor(mom[3], mt, hel)
            else:
                A, B = arg(w1, var), arg(w2, var)
                kA, kB = K[(w0 >> 16) & 0xFF], K[(w0 >> 24) & 0xFF]
                if op == 3:
                    r = (ir.mdot(A, B) * (kA - kB) + ir.mdot(2 * kB + kA, A) * B - ir.mdot(2 * kA + kB, B) * A) / ir.mdot(kout, kout)
                elif op == 4:
                    Z = arg(w3, var)
                    r = (ir.mdot(A, Z) * B - ir.mdot(B, Z) * A) / ir.mdot(kout, kout)
                elif op == 5:
                    q = -kout
                    r = A @ ir.slash(B) @ (ir.slash(q) + mt * np.eye(4)) / (ir.mdot(q, q) - mt * mt + 1j * mt * wt)
                elif op == 6:
                    q = kout
                    r = (ir.slash(q) + mt * np.eye(4)) @ ir.slash(A) @ B / (ir.mdot(q, q) - mt * mt + 1j * mt * wt)
                elif op == 7:
                    r = np.array([A @ ir.GAM[mu] @ B for mu in range(4)]) / ir.mdot(kout, kout)
                else:
                    raise ValueError(op)
            acc = acc + (-r if neg else r)
        obj.store(16 * (slot0 + _perm(var)), acc)

    nh = 1 << npar
    J = np.full((T["ncolor"], nh), np.nan + 0j, dtype=complex)
    for g in range(T["ngroups"]):
        stage = _Planes(T["stage_plane"])
        u0, nu, f0, nf = (int(x) for x in T["grp"][g])
        # phase 2: the units of the group (work items; each keeps its accumulators from one chunk to the next)
        for u in range(u0, u0 + nu):
            c0, nc = (int(x) for x in T["p2unit"][u])
            acc = np.zeros((32, 4), dtype=complex)
            for c in range(c0, c0 + nc):
                blk = T["p2rec"][c]
                for lane in range(32):
                    r0x, r0y = int(blk[0, lane, 0]), int(blk[0, lane, 1])
                    ctype, first, last = r0y & 0xFFF, (r0y >> 12) & 1, (r0y >> 13) & 1
                    if first:
                        acc[lane] = 0
                    for j in range(3):
                        op7 = (ctype >> (4 * j)) & 0xF
                        if op7 == 0:
                            break
                        op = op7 + 7
                        x, y = int(blk[1 + j, lane, 0]), int(blk[1 + j, lane, 1])
                        A, B = obj.load(x & 0xFFFF), obj.load(x >> 16)
                        Z = kA = kB = None
                        if op == 11:
                            assert (y & 0xFFFF) % 32 == 0 and (y >> 16) % 32 == 0
                            kA, kB = K[(y & 0xFFFF) // 32], K[(y >> 16) // 32]
                        elif op in (12, 13):
                            Z = obj.load(y & 0xFFFF)
                        r = _x_term(op, A, B, Z, kA, kB)
                        acc[lane] += -r if (r0x >> (16 + j)) & 1 else r
                    if last:
                        stage.store(r0x & 0xFFFF, acc[lane])
        # phase 3: the colour flows of the group (work items)
        if True:
            for f in range(f0, f0 + nf):
                rec0, info, cls0, jamp = (int(x) for x in T["p3flow"][f])
                ncls, nent = info & 0xFF, (info >> 8) & 0xFF
                accum = np.zeros(nh, dtype=complex)            # the flow's accumulator in shared memory, [slot]
                written = np.zeros(nh, dtype=bool)
                codes = T["p3shape_codes"]
                sig = [hs for hs, i in T["flow_sigs"].items() if i == (info >> 24) & 0x7F][0]      # slots per class
                assert ncls == len(sig)
                e = rec0
                for cls in range(cls0, cls0 + ncls):
                    hdr = int(T["p3clsh"][cls])
                    hslots = sig[cls - cls0]
                    frag = np.zeros((32, ntile), dtype=complex)    # register fragments of the class
                    nreal = 0
                    for k, code in enumerate(codes):               # the slots of shape k, in the kernel's order
                        for _ in range((hslots >> (4 * k)) & 15):
                            rec = T["p3rec"][e]
                            e += 1
                            flags = int(rec[0, 3])
                            assert all(int(rec[r, 3]) == flags for r in range(8))
                            if flags & 0x100:                      # slot not used by this flow
                                continue
                            assert (flags & 0xF) == code and hdr != 0
                            nreal += 1
                            neg = (flags >> 31) & 1
                            swapped, mask = code & 1, code >> 1
                            na = 1 << bin(mask).count("1")
                            nb = ntile // na
                            aplanes, bplanes = (obj, stage) if swapped else (stage, obj)
                            for lane in range(32):
                                # the MMA sums over the component index lane % 4 of the fragments; emulate it by letting lane
                                # (row r_, complex column c2) gather all four components of both operands itself
                                r_, c2 = lane >> 2, lane & 3
                                for t in range(ntile):
                                    ai = sum(((t >> b_) & 1) << i for i, b_ in enumerate([b_ for b_ in range(8) if (mask >> b_) & 1]))
                                    bi = sum(((t >> b_) & 1) << i for i, b_ in
                                             enumerate([b_ for b_ in range(ntile.bit_length() - 1) if not (mask >> b_) & 1]))
                                    arow = [int(x) for x in rec[r_, :3]]
                                    ah = [w_ >> (16 * q) & 0xFFFF for w_ in arow for q in range(2)][:na]
                                    # column c2 is served by record rows 2 c2 (re half) and 2 c2 + 1 (im half): same slot, +8 bytes
                                    brow = [int(x) for x in rec[2 * c2, :3]]
                                    bh = [w_ >> (16 * q) & 0xFFFF for w_ in brow for q in range(2)][2 * ((na + 1) // 2):][:nb]
                                    brow1 = [int(x) for x in rec[2 * c2 + 1, :3]]
                                    bh1 = [w_ >> (16 * q) & 0xFFFF for w_ in brow1 for q in range(2)][2 * ((na + 1) // 2):][:nb]
                                    assert bh[bi] % 16 == 0 and bh1[bi] == bh[bi] + 8
                                    val = np.sum(aplanes.load(ah[ai]) * bplanes.load(bh[bi]))
                                    frag[lane, t] += -val if neg else val
                    assert nreal == sum((hdr >> (4 * k)) & 15 for k in range(4))
                    if hdr == 0:                                   # class not used by this flow: the kernel skips its flush
                        continue
                    for lane in range(32):
                        for t in range(ntile):
                            off = int(T["p3cls"][cls][lane, t])
                            assert off % 16 == 0
                            accum[off // 16] += frag[lane, t]
                            written[off // 16] = True
                assert e == rec0 + nent and written.all()
                for h in range(nh):
                    J[jamp][h] = accum[_acc_swizzle(h)]
    assert not np.isnan(J).any()
    return J
