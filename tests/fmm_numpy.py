"""The translation formulas of the 2-D Stokeslet fast multipole method, written out with numpy (slow, small cases only).

Test infrastructure: an independent statement of what csrc/vn_fmm.cu implements (moments, M2M, M2L, L2L in variables
scaled by the box size, local evaluation, direct part over neighbour leaves, own-vesicle exclusion), used by
tests/test_fmm_formulas.py to check on the CPU that these formulas converge to the oracle's direct sum as the order
grows.  Complex notation: z = x + i y, g = gx + i gy;  u = -(Re Phi1 + i Re Phi2) + (z/2) conj(Phi1' + i Phi2') -
(1/2) conj(psi)  (see test_complex_potential_form_of_the_stokeslet_sum)."""
import numpy as np
from math import comb, log


def fmm(X, G, ves, L, p):
    z = X[:, 0] + 1j * X[:, 1]; g = G[:, 0] + 1j * G[:, 1]
    lo = X.min(0); size = (X.max(0) - lo).max() * (1 + 1e-9)
    n = 1 << L; s = size / n
    ix = np.minimum(((X[:, 0] - lo[0]) / s).astype(int), n - 1); iy = np.minimum(((X[:, 1] - lo[1]) / s).astype(int), n - 1)
    ctr = lambda l, i, j: (lo[0] + (i + 0.5) * size / (1 << l)) + 1j * (lo[1] + (j + 0.5) * size / (1 << l))
    K = np.arange(p + 1)
    # P2M
    A1 = [np.zeros((1 << l, 1 << l, p + 1), complex) for l in range(L + 1)]
    A2 = [np.zeros((1 << l, 1 << l, p + 1), complex) for l in range(L + 1)]
    B = [np.zeros((1 << l, 1 << l, p + 1), complex) for l in range(L + 1)]
    w = (z - ctr(L, ix, iy)) / s
    pw = w[:, None] ** K[None, :]
    np.add.at(A1[L], (ix, iy), g.real[:, None] * pw)
    np.add.at(A2[L], (ix, iy), g.imag[:, None] * pw)
    np.add.at(B[L], (ix, iy), (np.conj(z) * g)[:, None] * pw)
    # M2M
    S = np.zeros((4, p + 1, p + 1), complex)   # shift matrices for the four children
    deltas = {}
    for a in range(2):
        for b in range(2):
            d = ((a - 0.5) + 1j * (b - 0.5)) * 0.5
            deltas[(a, b)] = d
            for k in range(p + 1):
                for m in range(k + 1):
                    S[2 * a + b, k, m] = comb(k, m) * d ** (k - m) * 0.5 ** m
    for l in range(L, 0, -1):
        for arr in (A1, A2, B):
            for a in range(2):
                for b in range(2):
                    arr[l - 1] += np.einsum("km,ijm->ijk", S[2 * a + b], arr[l][a::2, b::2])
    # M2L
    b1 = [np.zeros((1 << l, 1 << l, p + 1), complex) for l in range(L + 1)]
    b2 = [np.zeros((1 << l, 1 << l, p + 1), complex) for l in range(L + 1)]
    dd = [np.zeros((1 << l, 1 << l, p + 1), complex) for l in range(L + 1)]
    for l in range(2, L + 1):
        nl = 1 << l; sl = size / nl
        for i in range(nl):
            for j in range(nl):
                pi, pj = i >> 1, j >> 1
                for si in range(max(0, 2 * (pi - 1)), min(nl, 2 * (pi + 1) + 2)):
                    for sj in range(max(0, 2 * (pj - 1)), min(nl, 2 * (pj + 1) + 2)):
                        if abs(si - i) <= 1 and abs(sj - j) <= 1: continue
                        a1, a2, bb = A1[l][si, sj], A2[l][si, sj], B[l][si, sj]
                        if a1[0] == 0 and a2[0] == 0 and not bb.any(): continue
                        tau = (i - si) + 1j * (j - sj)
                        for arr, out in ((a1, b1), (a2, b2)):
                            o = out[l][i, j]
                            o[0] += arr[0] * (log(sl) + np.log(tau)) - sum(arr[k] / (k * tau ** k) for k in range(1, p + 1))
                            for q in range(1, p + 1):
                                o[q] += arr[0] * (-1) ** (q + 1) / (q * tau ** q) - sum(arr[k] * comb(k + q - 1, q) * (-1) ** q / (k * tau ** (k + q)) for k in range(1, p + 1))
                        o = dd[l][i, j]
                        for q in range(p + 1):
                            o[q] += sum(bb[k] * comb(k + q, q) * (-1) ** q / tau ** (k + q + 1) for k in range(p + 1)) / sl
                        o[0] -= np.conj(a1[0] + 1j * a2[0])          # the constant g/2 of every far source
        # L2L to children
        if l < L:
            T = np.zeros((4, p + 1, p + 1), complex)
            for a in range(2):
                for b in range(2):
                    d = deltas[(a, b)]
                    for m in range(p + 1):
                        for q in range(m, p + 1):
                            T[2 * a + b, m, q] = 0.5 ** m * comb(q, m) * d ** (q - m)
            for arr in (b1, b2, dd):
                for a in range(2):
                    for b in range(2):
                        arr[l + 1][a::2, b::2] += np.einsum("mq,ijq->ijm", T[2 * a + b], arr[l])
    # L2P
    t = (z - ctr(L, ix, iy)) / s
    pt = t[:, None] ** K[None, :]
    Phi1 = np.sum(b1[L][ix, iy] * pt, 1); Phi2 = np.sum(b2[L][ix, iy] * pt, 1)
    dpt = np.zeros_like(pt); dpt[:, 1:] = K[None, 1:] * t[:, None] ** (K[None, 1:] - 1)
    dPhi1 = np.sum(b1[L][ix, iy] * dpt, 1) / s; dPhi2 = np.sum(b2[L][ix, iy] * dpt, 1) / s
    psi = np.sum(dd[L][ix, iy] * pt, 1)
    u = -(Phi1.real + 1j * Phi2.real) + 0.5 * z * np.conj(dPhi1 + 1j * dPhi2) - 0.5 * np.conj(psi)
    # P2P (neighbour boxes, other vesicles) and own-vesicle far correction
    order = np.lexsort((iy, ix)); 
    from collections import defaultdict
    cells = defaultdict(list)
    for idx in range(len(z)): cells[(ix[idx], iy[idx])].append(idx)
    for (ci, cj), tg in cells.items():
        src = []
        for a in range(ci - 1, ci + 2):
            for b in range(cj - 1, cj + 2):
                src += cells.get((a, b), [])
        src = np.array(src); tg = np.array(tg)
        r = z[tg][:, None] - z[src][None, :]
        mask = ves[tg][:, None] != ves[src][None, :]
        with np.errstate(divide="ignore", invalid="ignore"):
            term = -np.log(np.abs(r)) * g[src][None, :] + 0.5 * g[src][None, :] + 0.5 * (r / np.conj(r)) * np.conj(g[src])[None, :]
        u[tg] += np.where(mask, term, 0).sum(1)
    # own vesicle sources that sit in NON-neighbour boxes were summed through the expansions: take them out
    for v in np.unique(ves):
        idx = np.flatnonzero(ves == v)
        r = z[idx][:, None] - z[idx][None, :]
        far = (np.abs(ix[idx][:, None] - ix[idx][None, :]) > 1) | (np.abs(iy[idx][:, None] - iy[idx][None, :]) > 1)
        with np.errstate(divide="ignore", invalid="ignore"):
            term = -np.log(np.abs(r)) * g[idx][None, :] + 0.5 * g[idx][None, :] + 0.5 * (r / np.conj(r)) * np.conj(g[idx])[None, :]
        u[idx] -= np.where(far, term, 0).sum(1)
    return u
