"""tests/exact_interp.py — TEST INFRASTRUCTURE: exact rational evaluation (fractions.Fraction) of the integrand
from the product's device tables. The integrand is a rational function of z with rational coefficients, and a
double z is a rational number, so this is the exact value: it pins the oracle's binary128 result and the CUDA
double-double result without any floating-point arithmetic. Slow; tiny point sets only."""
from fractions import Fraction as Fr

from blob_interp import NGRADE, Blob, pairings


class ExactBlob(Blob):
    def scalars(self, g, z):
        n, ns = int(g["nch"]), int(g["nslot"])
        A = [[Fr(0)]*n for _ in range(n)]
        eps = [[(int(g["slot"][s]["eps"]) >> i) & 1 for i in range(n)] for s in range(ns)]
        for s in range(ns):
            if g["slot"][s]["kind"] == 0:
                zt = z[g["slot"][s]["zline"]]
                for i in range(n):
                    for j in range(n):
                        if eps[s][i] and eps[s][j]: A[i][j] += zt
        for i in range(n): A[i][i] += z[g["chord_zline"][i]]
        # exact Gauss-Jordan
        M = [row[:] + [Fr(int(i==j)) for j in range(n)] for i,row in enumerate(A)]
        det = Fr(1)
        for c in range(n):
            p = M[c][c]; det *= p
            M[c] = [v/p for v in M[c]]
            for r in range(n):
                if r != c and M[r][c] != 0:
                    f = M[r][c]; M[r] = [a - f*b for a,b in zip(M[r], M[c])]
        Inv = [row[n:] for row in M]
        beta = [[sum(Inv[i][j] for i in range(n) if eps[s][i] for j in range(n) if eps[u][j]) for u in range(ns)] for s in range(ns)]
        oat, oaq, obt = int(g["off_at"]), int(g["off_aq"]), int(g["off_bt"])
        S = [Fr(0)]*int(g["scal_len"]); ig=[Fr(1)]*ns; V=Fr(0); G=Fr(1)
        for s in range(ns):
            x=q=Fr(0)
            for u in range(ns):
                if g["slot"][u]["kind"]==0:
                    zb = beta[s][u]*z[g["slot"][u]["zline"]]; x+=zb; q+=zb*int(g["slot"][u]["sgn"])
            line = g["slot"][s]["kind"]==0
            gs = 2-x; ig[s] = 1/gs if line else Fr(1)
            S[s]=x*ig[s]
            if oat >= 0: S[oat+s]=1-x
            if oaq >= 0: S[oaq+s]=(int(g["slot"][s]["sgn"])-q)*ig[s]/2
            if line: V+=x*z[g["slot"][s]["zline"]]; G*=gs
        for s in range(ns):
            for u in range(s+1,ns): S[obt+s*ns-s*(s+1)//2+(u-s-1)] = beta[s][u]*ig[s]*ig[u]
        return S, det, V, G
    def family_value(self, c, kd, bidx, ridx, coef, S):
        n2=2*c
        if c not in self._pair_cache: self._pair_cache[c]=pairings(n2)
        b=[S[i] for i in bidx]; r=[S[i] for i in ridx]; tot=Fr(0); pos=0
        for pr in self._pair_cache[c]:
            w=Fr(1)
            for (i,j) in pr: w*=b[i*n2-i*(i+1)//2+(j-i-1)]
            blk=coef[pos:pos+(1<<kd)]; pos+=1<<kd
            if kd==0: h=Fr(float(blk[0]))
            else:
                half=1<<(kd-1); cc=[0]*(1<<kd)
                for j in range(half): cc[j]=blk[2*j]; cc[j+half]=blk[2*j+1]
                h=Fr(0)
                for sig in range(1<<kd):
                    if cc[sig]==0: continue
                    m=Fr(float(cc[sig]))
                    for i in range(kd):
                        if sig>>i&1: m*=r[i]
                    h+=m
            tot+=w*h
        return tot
    def integrand(self, z):
        h=self.h; nodeval,nodeU,nodeV={},{},{}
        def conv(a,b):
            out=[Fr(0)]*NGRADE
            for i in range(NGRADE):
                for j in range(NGRADE-i): out[i+j]+=a[i]*b[j]
            return out
        for gi in range(int(h["ngeom"])):
            g=self.geom[gi]; S,U,V,G=self.scalars(g,z); npat=1<<int(g["nS"])
            for ti in range(int(g["first_table"]), int(g["first_table"]+g["ntable"])):
                t=self.table[ti]; N=[[[Fr(0)]*NGRADE for _ in range(npat)] for _ in range(2)]
                for (c,kd,pat,out,bidx,ridx,sidx,coef) in self.families(ti):
                    val=self.family_value(c,kd,bidx,ridx,coef,S)
                    for i in sidx: val*=S[i]
                    N[out][pat][c]+=val
                if int(t["nout"])==1 and int(t["op"]) in (1,3):
                    N[0]=[[v/12 for v in row] for row in N[0]]
                for ni in range(int(t["first_node"]), int(t["first_node"]+t["nnode"])):
                    nd=self.node[ni]; Up,Vs=U,V
                    for k in range(int(nd["nchild"])): Up*=nodeU[int(nd["child"][k])]; Vs+=nodeV[int(nd["child"][k])]
                    nodeU[ni],nodeV[ni]=Up,Vs; vals=[[Fr(0)]*NGRADE for _ in range(2)]
                    for o in range(int(nd["nout"])):
                        for p in range(npat):
                            acc=[v*G for v in N[o][p]]
                            for k in range(int(nd["nchild"])):
                                pb=int(g["child_patbit"][k]); which=1 if (pb>=0 and (p>>pb&1)) else 0
                                acc=conv(acc,nodeval[int(nd["child"][k])][which])
                            vals[o]=[a+b for a,b in zip(vals[o],acc)]
                    nodeval[ni]=vals
        L=int(h["L"]); f=Fr(0)
        for t in self.term:
            root=int(t["root"]); U2=nodeU[root]**2; Vs=nodeV[root]; fact=1
            for c in range(L-1,-1,-1):
                if L-c-1>0: fact*=L-c-1
                f+=int(t["sign"])*fact*nodeval[root][0][c]/(U2*Vs**(L-c))
        return f
