"""tests/blob_interp.py — TEST INFRASTRUCTURE: a slow pure-Python reader of the device table blob
(paper_1905_08007_b200/csrc/device_layout.h). It lets the CPU test-suite check the product's host
preparation (numerator tables, term trees, sampler tables) against the oracle without a GPU.
It is not a fallback: nothing in the product imports it.
"""
import itertools

import numpy as np

MAXL, MAXSLOT, MAXCHILD, NGRADE = 5, 14, 5, 6
HDR = np.dtype([("L", "<i4"), ("M", "<i4"), ("diag_id", "<i4"), ("ngeom", "<i4"), ("ntable", "<i4"), ("nnode", "<i4"), ("nterm", "<i4"),
                ("nodeval_len", "<i4"), ("max_scal_len", "<i4"), ("wl", "<i4"), ("C", "<f8"), ("cond_max", "<f8"),
                ("off_Z", "<i8"), ("off_invdeg", "<i8"), ("off_geom", "<i8"), ("off_table", "<i8"), ("off_node", "<i8"), ("off_term", "<i8"), ("total_words", "<i8"),
                ("off_stream", "<i8"), ("stream_chunks", "<i8"), ("rng", "<i4"), ("pad0", "<i4"), ("off_mrg", "<i8"),
                ("mix_alpha", "<f8"), ("C2", "<f8"), ("off_Z2", "<i8"), ("off_invdeg2", "<i8"), ("off_deg1", "<i8"), ("off_deg2", "<i8")])
SLOT = np.dtype([("kind", "i1"), ("zline", "i1"), ("sgn", "i1"), ("child", "i1"), ("eps", "<u4")])
GEOM = np.dtype([("nch", "<i4"), ("nslot", "<i4"), ("nchild", "<i4"), ("nS", "<i4"), ("chord_zline", "<i4", (MAXL,)), ("slot", SLOT, (MAXSLOT,)),
                 ("child_type", "i1", (MAXCHILD,)), ("child_patbit", "i1", (MAXCHILD,)), ("pad", "<i2"), ("first_table", "<i4"), ("ntable", "<i4"),
                 ("off_at", "<i4"), ("off_aq", "<i4"), ("off_bt", "<i4"), ("scal_len", "<i4")])
TABLE = np.dtype([("geom", "<i4"), ("op", "<i4"), ("nout", "<i4"), ("nfam", "<i4"), ("first_node", "<i4"), ("nnode", "<i4"),
                  ("stream_off", "<i8"), ("stream_words", "<i8"), ("n_monomials", "<i8")])
NODE = np.dtype([("table", "<i4"), ("geom", "<i4"), ("nchild", "<i4"), ("nout", "<i4"), ("child", "<i4", (MAXCHILD,)), ("val_off", "<i4"), ("ngr", "<i4")])
TERM = np.dtype([("root", "<i4"), ("sign", "<i4")])
assert GEOM.itemsize == 184 and TABLE.itemsize == 48 and NODE.itemsize == 44 and HDR.itemsize == 192


def pairings(n2):
    """canonical order: the first free element pairs with every later one"""
    def rec(free):
        if not free:
            yield []
            return
        f = free[0]
        for s in free[1:]:
            rest = [x for x in free if x != f and x != s]
            for tail in rec(rest):
                yield [(f, s)] + tail
    return list(rec(list(range(n2))))


def _flatten_big_blocks(coef, kd):
    """device_layout.h: a kd = 5, 6 block is stored as 2^(kd-4) sub-blocks of kd = 4, each as units (c[j], c[j+8]); returns the
    block in the single-level layout (c[j], c[j+2^(kd-1)]) that family_value undoes"""
    n, half = 1 << kd, 1 << (kd - 1)
    out = np.empty_like(coef)
    for q in range(len(coef) // n):
        blk = coef[q * n:(q + 1) * n]
        nat = np.empty(n)
        for top in range(n >> 4):
            sub = blk[top * 16:(top + 1) * 16]
            nat[(top << 4):(top << 4) + 8] = sub[0::2]
            nat[(top << 4) + 8:(top << 4) + 16] = sub[1::2]
        o = out[q * n:(q + 1) * n]
        o[0::2], o[1::2] = nat[:half], nat[half:]
    return out


class Blob:
    def __init__(self, words):
        self.w = np.ascontiguousarray(words, np.uint64)
        raw = self.w.view(np.uint8)
        self.h = np.frombuffer(raw, HDR, 1)[0]
        h = self.h
        self.Z = self.w[h["off_Z"]:h["off_Z"] + (1 << h["M"])].view(np.float64)
        self.invdeg = self.w[h["off_invdeg"]:h["off_invdeg"] + (1 << h["M"])].view(np.float64)
        self.geom = np.frombuffer(raw, GEOM, h["ngeom"], h["off_geom"] * 8)
        self.table = np.frombuffer(raw, TABLE, h["ntable"], h["off_table"] * 8)
        self.node = np.frombuffer(raw, NODE, h["nnode"], h["off_node"] * 8)
        self.term = np.frombuffer(raw, TERM, h["nterm"], h["off_term"] * 8)
        self._pair_cache = {}

    def families(self, ti):
        """yields the families of table ti; a stream entry holds WL same-shape families side by side (device_layout.h)"""
        WL = int(self.h["wl"])
        t = self.table[ti]
        pos = int(t["stream_off"])
        raw = self.w.view(np.uint8)
        nleft = int(t["nfam"])                       # stream entries
        while nleft:
            hd = int(self.w[pos])
            c, kd = hd & 7, hd >> 3 & 7
            idxw, ncoef = hd >> 16 & 0xFFFF, hd >> 32 & 0xFFFF
            if c == 7:                      # PAD entry up to the chunk boundary
                pos += 1 + idxw
                continue
            nleft -= 1
            nb = c * (2 * c - 1)
            assert ncoef % WL == 0 and (pos + WL * (1 + idxw)) % 2 == 0
            unit = 2 if kd >= 1 else 1
            allc = self.w[pos + WL * (1 + idxw):pos + WL * (1 + idxw) + ncoef].view(np.float64).reshape(-1, WL, unit)
            for m in range(WL):
                hm = int(self.w[pos + m])
                assert (hm & 63) == (hd & 63) and (hm >> 16) == (hd >> 16)
                pat, nscal, out, void = hm >> 6 & 15, hm >> 10 & 15, hm >> 14 & 1, hm >> 15 & 1
                coef = np.ascontiguousarray(allc[:, m, :]).reshape(-1)
                if kd >= 3:                     # strip (and check) the closing (sum |c|, 0) unit of every block
                    blocks = coef.reshape(-1, (1 << kd) + 2)
                    assert np.array_equal(blocks[:, -2], np.abs(blocks[:, :-2]).sum(axis=1)) and not blocks[:, -1].any()
                    coef = np.ascontiguousarray(blocks[:, :-2]).reshape(-1)
                if kd > 4:                      # sub-blocks of kd = 4 (top index bits ascending) -> one (lo,hi)-interleaved block
                    coef = _flatten_big_blocks(coef, kd)
                if void:
                    assert not coef.any()
                    continue
                at = (pos + WL + m * idxw) * 8
                idx = raw[at:at + nb + kd + nscal].astype(int)
                yield c, kd, pat, out, idx[:nb], idx[nb:nb + kd], idx[nb + kd:], coef
            pos += WL * (1 + idxw) + ncoef
        assert pos == int(t["stream_off"] + t["stream_words"])

    def scalars(self, g, z):
        n, ns = int(g["nch"]), int(g["nslot"])
        A = np.zeros((n, n))
        eps = [[(int(g["slot"][s]["eps"]) >> i) & 1 for i in range(n)] for s in range(ns)]
        for s in range(ns):
            if g["slot"][s]["kind"] == 0:
                e = np.array(eps[s], float)
                A += z[g["slot"][s]["zline"]] * np.outer(e, e)
        for i in range(n):
            A[i, i] += z[g["chord_zline"][i]]
        U = np.linalg.det(A)
        Inv = np.linalg.inv(A)
        E = np.array(eps, float).reshape(ns, n)
        beta = E @ Inv @ E.T
        oat, oaq, obt = int(g["off_at"]), int(g["off_aq"]), int(g["off_bt"])
        S = np.zeros(int(g["scal_len"]))
        ig = np.ones(ns)
        V, G = 0.0, 1.0
        for s in range(ns):
            x = q = 0.0
            for u in range(ns):
                if g["slot"][u]["kind"] == 0:
                    zb = beta[s, u] * z[g["slot"][u]["zline"]]
                    x += zb
                    q += zb * g["slot"][u]["sgn"]
            line = g["slot"][s]["kind"] == 0
            gs = 2.0 - x
            ig[s] = 1.0 / gs if line else 1.0
            S[s] = x * ig[s]
            if oat >= 0:
                S[oat + s] = 1.0 - x
            if oaq >= 0:
                S[oaq + s] = (g["slot"][s]["sgn"] - q) * ig[s] * 0.5
            if line:
                V += x * z[g["slot"][s]["zline"]]
                G *= gs
        for s in range(ns):
            for u in range(s + 1, ns):
                S[obt + s * ns - s * (s + 1) // 2 + (u - s - 1)] = beta[s, u] * ig[s] * ig[u]
        return S, U, V, G

    def family_value(self, c, kd, bidx, ridx, coef, S):
        n2 = 2 * c
        if c not in self._pair_cache:
            self._pair_cache[c] = pairings(n2)
        b = S[bidx] if len(bidx) else np.zeros(0)
        r = S[ridx] if len(ridx) else np.zeros(0)
        tot, pos = 0.0, 0
        for pr in self._pair_cache[c]:
            w = 1.0
            for (i, j) in pr:
                w *= b[i * n2 - i * (i + 1) // 2 + (j - i - 1)]
            blk = coef[pos:pos + (1 << kd)]
            pos += 1 << kd
            if kd == 0:
                h = blk[0]
            else:
                half = 1 << (kd - 1)
                cc = np.empty(1 << kd)
                cc[:half], cc[half:] = blk[0::2], blk[1::2]       # undo the (lo,hi) interleave
                h = 0.0
                for sig in range(1 << kd):
                    m = cc[sig]
                    for i in range(kd):
                        if sig >> i & 1:
                            m *= r[i]
                    h += m
            tot += w * h
        assert pos == len(coef)
        return tot

    def integrand(self, z):
        h = self.h
        nodeval, nodeU, nodeV = {}, {}, {}
        for gi in range(int(h["ngeom"])):
            g = self.geom[gi]
            S, U, V, G = self.scalars(g, z)
            npat = 1 << int(g["nS"])
            for ti in range(int(g["first_table"]), int(g["first_table"] + g["ntable"])):
                t = self.table[ti]
                N = np.zeros((2, npat, NGRADE))
                for (c, kd, pat, out, bidx, ridx, sidx, coef) in self.families(ti):
                    val = self.family_value(c, kd, bidx, ridx, coef, S)
                    for i in sidx:
                        val *= S[i]
                    N[out, pat, c] += val
                if int(t["nout"]) == 1 and int(t["op"]) in (1, 3):      # U, L-U on a vertex-like piece: table holds 12*coef
                    N[0] /= 12.0
                for ni in range(int(t["first_node"]), int(t["first_node"] + t["nnode"])):
                    nd = self.node[ni]
                    Up, Vs = U, V
                    for k in range(int(nd["nchild"])):
                        Up *= nodeU[int(nd["child"][k])]
                        Vs += nodeV[int(nd["child"][k])]
                    nodeU[ni], nodeV[ni] = Up, Vs
                    vals = np.zeros((2, NGRADE))
                    for o in range(int(nd["nout"])):
                        for p in range(npat):
                            acc = N[o, p] * G
                            for k in range(int(nd["nchild"])):
                                pb = int(g["child_patbit"][k])
                                which = 1 if (pb >= 0 and (p >> pb & 1)) else 0
                                acc = np.convolve(acc, nodeval[int(nd["child"][k])][which])[:NGRADE]
                            vals[o] += acc
                    nodeval[ni] = vals
        L = int(h["L"])
        f, terms = 0.0, []
        for t in self.term:
            root = int(t["root"])
            U2, Vs = nodeU[root] ** 2, nodeV[root]
            ft, fact = 0.0, 1.0
            for c in range(L - 1, -1, -1):
                if L - c - 1 > 0:
                    fact *= L - c - 1
                ft += int(t["sign"]) * fact * nodeval[root][0][c] / (U2 * Vs ** (L - c))
            terms.append(ft)
            f += ft
        return f, terms
