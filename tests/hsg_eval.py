"""numpy interpreter of the tables of the generic helicity-shared kernel (gen/hsg_tables.py) -- CPU TEST HELPER.

Executes what one CTA of csrc/hsg_kernel.cu executes for one event from the same packed tables (objects, pair objects,
entries, variant lookup); every opcode is restated with the plain gamma-matrix helpers of tests/ir_eval.py.  So the
generator's factorisation at 6 gluons (4-leg colour-ordered objects, the X.Y split and its signs, the packing) is checked
against the oracle on CPU before any kernel runs.  Not product, not oracle; nothing here is imported by the package.
"""
import numpy as np

import ir_eval as ir

G = ir.G


def _sub(v, code):
    return sum(((v >> ((code >> (3 * j)) & 7)) & 1) << j for j in range(4))


def _x_term(op, A, B, Z, kA, kB):
    if op == 8:
        return A @ ir.slash(B)
    if op == 9:
        return ir.slash(A) @ B
    if op == 10:
        return np.array([A @ ir.GAM[mu] @ B for mu in range(4)])
    if op == 11:
        return ir.mdot(A, B) * (kA - kB) + ir.mdot(2 * kB + kA, A) * B - ir.mdot(2 * kA + kB, B) * A
    if op == 12:
        return ir.mdot(A, Z) * B - ir.mdot(B, Z) * A
    if op == 13:
        return 2 * ir.mdot(A, Z) * B - ir.mdot(B, Z) * A - ir.mdot(A, B) * Z
    raise ValueError(op)


def _area(T, mom, mt, wt):
    """phases 1 and 2: the scratch area of one event, [slot][component]"""
    npar = T["npar"]
    k = [mom[i] * (1 if i < 2 else -1) for i in range(npar)]
    K = [sum(k[p] for p in range(npar) if (m >> p) & 1) for m in T["legset_mask"]]
    area = np.full((T["nslot"], 4), np.nan + 0j, dtype=complex)

    def arg(w, var):
        return area[(w & 0xFFFF) + _sub(var, (w >> 16) & 0xFFF)]

    for it in T["p1_items"]:
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
        assert np.isnan(area[slot0 + var]).all()
        area[slot0 + var] = acc

    for a, b in T["xitem"]:
        a, b = int(a) & 0xFFFFFFFF, int(b) & 0xFFFFFFFF
        t0, nt = a & 0xFFFFFF, a >> 24
        slot, var, vec = b & 0xFFFFF, (b >> 20) & 0xFF, (b >> 28) & 1
        acc = np.zeros(4, dtype=complex)
        for t in T["term"][t0:t0 + nt]:
            w0, w1, w2, w3 = (int(x) & 0xFFFFFFFF for x in t)
            op, neg = w0 & 0xFF, (w0 >> 8) & 1
            A, B = arg(w1, var), arg(w2, var)
            Z = arg(w3, var) if op in (12, 13) else None
            r = _x_term(op, A, B, Z, K[(w0 >> 16) & 0xFF], K[(w0 >> 24) & 0xFF])
            assert (op >= 10) == bool(vec)
            acc = acc + (-r if neg else r)
        assert np.isnan(area[slot]).all()
        area[slot] = G * acc if vec else acc
    assert not np.isnan(area).any()
    return area


def evaluate(T, mom, mt, wt):
    """jamps[ncolor][2^npar] (without the g^n factor) of one event"""
    npar = T["npar"]
    area = _area(T, mom, mt, wt)
    nh = 1 << npar
    J = np.zeros((T["ncolor"], nh), dtype=complex)
    for j, e0, ne, _ in T["flow"]:
        for xs, ys, row, flags in T["entry"][e0:e0 + ne]:
            vt = T["vtab"][row].astype(np.int64)
            X = area[int(xs) + (vt & 0xFF)]
            Y = area[int(ys) + (vt >> 8)]
            J[j] += (-1 if int(flags) & 1 else 1) * np.sum(X * Y, axis=1)
            # bits 1..3: which of particles 0, 1, 2 are legs of X; they are the highest bits of the variant index of the object
            # that holds them (descending particle order), above its lx (ly) other legs (bits 4..6, 7..9)
            fl = int(flags)
            lx, ly = (fl >> 4) & 7, (fl >> 7) & 7
            for i in range(3):
                hbit = 1 << (npar - 1 - i)
                dx = (vt[hbit] & 0xFF) - (vt[0] & 0xFF)
                dy = (vt[hbit] >> 8) - (vt[0] >> 8)
                inx = (fl >> (1 + i)) & 1
                above = sum(1 for b in range(i + 1, 3) if ((fl >> (1 + b)) & 1) == inx)       # larger fixed particles sit below
                assert (dx, dy) == ((1 << (lx + above), 0) if inx else (0, 1 << (ly + above)))
    return J


def _acc_swz(h):
    """csrc/hsg_kernel.cu acc_swz, restated"""
    hi, g = h >> 3, 0
    for b, pat in enumerate((3, 5, 6, 7, 1)):
        if (hi >> b) & 1:
            g ^= pat
    return h ^ g


def evaluate_tensor(T, mom, mt, wt, flows=None):
    """the same jamps from the tables of the TENSOR path of phase 3 (dentry, ltab, flowL, flowT), executed the way a warp of
    csrc/hsg_kernel.cu executes them: the entry's operands copied into a byte-addressed buffer (X then Y: 4 component planes of
    2^lg + 1 slots of 16 bytes, variant bits 2 and swx / swy exchanged), fragments of mma.sync.m8n8k4.f64 gathered per lane from the table offsets (a = A[lane / 4][lane % 4],
    b = B[lane % 4][lane / 4], c0, c1 = C[lane / 4][2 (lane % 4) + {0, 1}]), two k-steps per tile into separate accumulators,
    classes flushed to the swizzled accumulator, read back in the order of the helicity combinations"""
    npar = T["npar"]
    assert npar == 8
    area = _area(T, mom, mt, wt)
    nh = 1 << npar
    J = np.zeros((T["ncolor"], nh), dtype=complex)
    lanes = np.arange(32)
    for f, (j, e0, ne, ncls) in enumerate(T["flow"]):
        if flows is not None and f not in flows:
            continue
        acc = np.full((nh, 2), np.nan)
        frag = np.zeros((8, 32, 4))
        cls = 0
        for k in range(e0, e0 + ne):
            w0, w1, w2, w3 = (int(x) & 0xFFFFFFFF for x in T["dentry"][k])
            xs, ys = w0 & 0xFFFF, w0 >> 16
            row, lgx, mask, neg, last = w1 & 0xFFFF, (w1 >> 16) & 0xF, (w1 >> 20) & 7, (w1 >> 23) & 1, (w1 >> 24) & 1
            assert (xs, ys) == (int(T["entry"][k][0]), int(T["entry"][k][1])) and neg == (int(T["entry"][k][3]) & 1)
            lgy = npar - lgx
            d = (w2 & 0xFFFF, w2 >> 16, w3 & 0xFFFF)
            swx, swy = (w3 >> 16) & 0xF, (w3 >> 20) & 0xF

            def swap2(v, sw):          # variant index with bits 2 and sw exchanged
                x = ((v >> 2) ^ (v >> sw)) & 1
                return v ^ (x << 2) ^ (x << sw)

            psx, psy = (16 << lgx) + 16, (16 << lgy) + 16
            buf = np.full((4 * psx + 4 * psy) // 8, np.nan)                      # doubles
            for c in range(4):
                for v in range(1 << lgx):
                    o = (c * psx + 16 * v) // 8
                    buf[o], buf[o + 1] = area[xs + swap2(v, swx), c].real, area[xs + swap2(v, swx), c].imag
                for v in range(1 << lgy):
                    o = (4 * psx + c * psy + 16 * v) // 8
                    buf[o], buf[o + 1] = area[ys + swap2(v, swy), c].real, area[ys + swap2(v, swy), c].imag
            lt = T["ltab"][row].astype(np.int64)
            aoff, boff = lt & 0xFFFF, lt >> 16
            sg = -1.0 if neg else 1.0
            for t in range(8):
                ao, bo = aoff.copy(), boff.copy()
                for i in range(3):
                    if (t >> i) & 1:
                        if (mask >> i) & 1:
                            ao += d[i]
                        else:
                            bo += d[i]
                assert (ao % 16 == 0).all() and (bo % 8 == 0).all()
                are, aim = buf[ao // 8], buf[ao // 8 + 1]
                b0, b1 = buf[bo // 8], buf[(bo ^ 8) // 8]
                A0, A1, B0, B1 = np.zeros((8, 4)), np.zeros((8, 4)), np.zeros((4, 8)), np.zeros((4, 8))
                A0[lanes >> 2, lanes & 3], A1[lanes >> 2, lanes & 3] = sg * are, sg * aim
                B0[lanes & 3, lanes >> 2], B1[lanes & 3, lanes >> 2] = b0, b1
                C0, C1 = A0 @ B0, A1 @ B1
                frag[t, :, 0] += C0[lanes >> 2, 2 * (lanes & 3)]
                frag[t, :, 1] += C0[lanes >> 2, 2 * (lanes & 3) + 1]
                frag[t, :, 2] += C1[lanes >> 2, 2 * (lanes & 3)]
                frag[t, :, 3] += C1[lanes >> 2, 2 * (lanes & 3) + 1]
            if last:
                L = (T["flowL"][f].astype(np.int64) >> (8 * cls)) & 0xFF
                tw = int(T["flowT"][f][2 * cls]) | (int(T["flowT"][f][2 * cls + 1]) << 32)
                for t in range(8):
                    idx = L ^ ((tw >> (8 * t)) & 0xFF)
                    add = np.stack([frag[t, :, 0] - frag[t, :, 2], frag[t, :, 1] + frag[t, :, 3]], axis=1)
                    if cls == 0:
                        assert np.isnan(acc[idx]).all()
                        acc[idx] = add
                    else:
                        acc[idx] += add
                frag[:] = 0.0
                cls += 1
        assert cls == ncls and not np.isnan(acc).any()
        for h in range(nh):
            J[j, h] = complex(*acc[_acc_swz(h)])
    return J
