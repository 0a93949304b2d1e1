"""numpy interpreter of the helicity-shared program tables (gen/co_program.py) -- CPU TEST HELPER.

Decodes the int32 tables exactly as csrc/hs_kernel.cu does (same packing, same variant convention) and
restates every opcode with the plain gamma-matrix helpers of tests/ir_eval.py, so that the generator's
factorised program can be checked against the diagram program and the oracle before any kernel runs.
Not product, not oracle; nothing here is imported by the package.
"""
import numpy as np

import ir_eval as ir

G = ir.G


def _sub(v, code):
    """variant of an argument: bit j = bit (code >> 3j) & 7 of the parent's variant (7 = none)"""
    return sum(((v >> ((code >> (3 * j)) & 7)) & 1) << j for j in range(3))


def evaluate(T, mom, mt, wt):
    """jamps[ncolor][2^npar] (without the g^n factor) of one event from the tables T"""
    npar = T["npar"]
    k = [mom[i] * (1 if i < 2 else -1) for i in range(npar)]
    K = [sum(k[p] for p in range(npar) if (m >> p) & 1) for m in T["legset_mask"]]
    obj, term = T["obj"], T["term"]
    area = np.zeros(T["obj_area"], dtype=complex)
    # this interpreter keeps an object as [variant][component]; the kernel's bank swizzle is not modelled

    def load(w, var):
        off, code = w & 0xFFFF, (w >> 16) & 0x1FF
        return area[off + 4 * _sub(var, code):off + 4 * _sub(var, code) + 4].copy()

    def run_terms(t0, nt, var, legs_of_parent=None, kout=None):
        acc = np.zeros(4, dtype=complex)
        for t in term[t0:t0 + nt]:
            w0, w1, w2, w3 = (int(x) & 0xFFFFFFFF for x in t)
            op, neg = w0 & 0xFF, (w0 >> 8) & 1
            a = [w1]
            hel = 1 if var & 1 else -1
            if op == 0:
                e = ir.polvec(mom[a[0]], hel)
                r = e if a[0] < 2 else e.conj()
            elif op == 1:
                r = ir.u_spinor(mom[2], mt, hel).conj() @ ir.GAM[0]
            elif op == 2:
                r = ir.v_spinor(mom[3], mt, hel)
            else:
                A = load(w1, var)
                B = load(w2, var)
                kA, kB = K[(w0 >> 16) & 0xFF], K[(w0 >> 24) & 0xFF]
                if op == 3:
                    r = (ir.mdot(A, B) * (kA - kB) + ir.mdot(2 * kB + kA, A) * B - ir.mdot(2 * kA + kB, B) * A) / ir.mdot(kout, kout)
                elif op == 4:
                    Z = load(w3, var)
                    r = (ir.mdot(A, Z) * B - ir.mdot(B, Z) * A) / ir.mdot(kout, kout)
                elif op == 5:
                    q = -kout
                    r = A @ ir.slash(B) @ (ir.slash(q) + mt * np.eye(4)) / (ir.mdot(q, q) - mt * mt + 1j * mt * wt)
                elif op == 6:
                    q = kout
                    r = (ir.slash(q) + mt * np.eye(4)) @ ir.slash(A) @ B / (ir.mdot(q, q) - mt * mt + 1j * mt * wt)
                elif op == 7:
                    r = np.array([A @ ir.GAM[mu] @ B for mu in range(4)]) / ir.mdot(kout, kout)
                elif op == 8:
                    r = A @ ir.slash(B)
                elif op == 9:
                    r = ir.slash(A) @ B
                elif op == 10:
                    r = G * np.array([A @ ir.GAM[mu] @ B for mu in range(4)])
                elif op == 11:
                    r = G * (ir.mdot(A, B) * (kA - kB) + ir.mdot(2 * kB + kA, A) * B - ir.mdot(2 * kA + kB, B) * A)
                elif op == 12:
                    Z = load(w3, var)
                    r = G * (ir.mdot(A, Z) * B - ir.mdot(B, Z) * A)
                elif op == 13:
                    Z = load(w3, var)
                    r = G * (2 * ir.mdot(A, Z) * B - ir.mdot(B, Z) * A - ir.mdot(A, B) * Z)
                else:
                    raise ValueError(op)
            acc = acc + (-r if neg else r)
        return acc

    # phase 1: objects, level by level
    for it in T["p1_items"]:
        o, var = int(it) >> 8, int(it) & 0xFF
        off, info, t0, nt = (int(x) for x in obj[o])
        val = run_terms(t0, nt, var, kout=K[info >> 8])
        area[off + 4 * var:off + 4 * var + 4] = val
    # phases 2 and 3, group by group
    nh = 1 << npar
    J = np.zeros((T["ncolor"], nh), dtype=complex)
    stage = np.zeros(max(T["stage_area"], 1), dtype=complex)
    for g in T["group"]:
        x0, xi0, nxi, s0, ns = (int(x) for x in g[:5])
        for it in T["x_items"][xi0:xi0 + nxi]:
            if int(it) < 0:                                   # padding of the last work unit
                continue
            xk, var = int(it) >> 8, int(it) & 0xFF
            soff, lognv, t0, nt = (int(x) for x in T["xobj"][x0 + xk])
            stage[soff + 4 * var:soff + 4 * var + 4] = run_terms(t0, nt, var)
        for sg in T["sigma"][s0:s0 + ns]:
            j, e0, ne = int(sg[0]), int(sg[1]), int(sg[2])
            for h in range(nh):
                acc = 0j
                for e in T["entry"][e0:e0 + ne]:
                    w0, w1, row, sign = (int(x) for x in e)
                    offx, nvx = w0 & 0xFFFF, w0 >> 16
                    offy, nvy = w1 & 0xFFFF, w1 >> 16
                    vv = int(T["vtab"][row][h])
                    vx, vy = vv & 0xFF, vv >> 8
                    d = sum(stage[offx + 4 * vx + c] * area[offy + 4 * vy + c] for c in range(4))
                    acc += sign * d
                J[j][h] = acc
    return J
