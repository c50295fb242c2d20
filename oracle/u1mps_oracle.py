"""CPU ORACLE (test infrastructure, NOT the product) for the charge-blocked two-site update of a
U(1)-symmetric matrix-product state, arXiv:2303.11409.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference leg may import
this file.  It shares no code with the CUDA path (paper_2303_11409_b200/csrc) and never imports it.

Plain numpy, complex128 / float64 (reading S12: the paper states no precision; BASELINE.json fixes
complex128).  Written sector by sector in the paper's order and notation so that it can be checked
against PAPER.md by eye:

  state      {Gamma^[k], lambda^[k], c^[k]}                      PAPER.md L108-114, Eq.15
  Theta(c)   sum over alpha_k of U-entry * lam Gam lam Gam lam   PAPER.md L116-121, Eq.16
  SVD        one LAPACK SVD per Theta(c^[k])                     PAPER.md L121, Eq.12
  truncate   chi largest singular values over ALL Theta(c)
  new Gamma  V / lambda^[k-1],  W / lambda^[k+1]                 PAPER.md L94-104, Eq.13/14

Readings of silent / garbled passages are the S-numbers of SURVEY.md §8(c), restated in DESIGN.md.

Indexing (0-based, as the C ABI): sites s = 0..M-1, bonds k = 0..M; site s has left bond s and
right bond s+1.  c^[k] = number of particles on sites k..M-1 (right of bond k; reading S2), so
bond 0 = {N}, bond M = {0} and the occupation of site s is c_left - c_right (Eq.15's delta, L114).

Pins (tests/test_oracle_pins.py, all `-m "not gpu"`): P1 exact state vector (M<=16), P2 charge
invariants, P3 unit norm, P4 canonical-form identities, P5 Eckart-Young reconstruction, P6 brute
force dense (non-symmetric) update Eq.11-14, P7 identity/swap gates, P8 closed forms (single
particle walk, permanents, Hong-Ou-Mandel), P9 free-fermion <n_k>, P10 readout formula vs full
environments, P11 tie order at the cut, P12 two-point <n_j n_k> vs the state vector, P13 Fock-pattern sampling vs conditional
probabilities summed over the state vector.  Every function below is reached by at least one of them; nothing is
"parity unpinned".
"""
from __future__ import annotations

import math
from dataclasses import dataclass, field
from typing import Dict, List, Tuple

import numpy as np

Block = Tuple[int, int]


@dataclass
class GateRecord:
    """Everything one two-site update produced, for teacher-forced comparison (SURVEY §8(c) parity protocol)."""
    site: int
    charges: List[int] = field(default_factory=list)          # candidate centre charges c, ascending
    rows: Dict[int, List[Tuple[int, int, int]]] = field(default_factory=dict)  # c -> [(c_l, offset, n)]
    cols: Dict[int, List[Tuple[int, int, int]]] = field(default_factory=dict)  # c -> [(c_r, offset, n)]
    theta: Dict[int, np.ndarray] = field(default_factory=dict)  # c -> Theta(c)
    V: Dict[int, np.ndarray] = field(default_factory=dict)
    sigma: Dict[int, np.ndarray] = field(default_factory=dict)  # c -> all singular values, descending
    W: Dict[int, np.ndarray] = field(default_factory=dict)
    keep: Dict[int, int] = field(default_factory=dict)          # c -> number kept
    weight_kept: float = 0.0
    weight_all: float = 0.0
    discarded: float = 0.0
    sigma_chi: float = 0.0       # smallest kept singular value (before renormalisation)
    sigma_next: float = 0.0      # largest singular value above the cutoff that was NOT kept (0 if none)
    cutoff_gap: float = math.inf  # min |sigma - cutoff| over the pool (near-tie detector for the cutoff)


class U1MPS:
    """U(1)-symmetric canonical (Vidal) MPS stored as dense blocks per charge sector."""

    def __init__(self, M: int, d: int, N: int, chi: int):
        self.M, self.d, self.N, self.chi = M, d, N, chi
        self.sectors: List[List[int]] = [[] for _ in range(M + 1)]           # bond k -> ascending charges
        self.lam: List[Dict[int, np.ndarray]] = [dict() for _ in range(M + 1)]   # bond k -> c -> lambda (desc)
        self.gam: List[Dict[Block, np.ndarray]] = [dict() for _ in range(M)]     # site s -> (c_l,c_r) -> block
        self.log_norm = 0.0
        self.discarded_total = 0.0

    # ---------------------------------------------------------------- state construction
    @classmethod
    def product_state(cls, M: int, d: int, N: int, chi: int, occ) -> "U1MPS":
        """|occ_0 ... occ_{M-1}>: every bond has one sector of multiplicity 1 (SURVEY §8(c) State)."""
        occ = [int(o) for o in occ]
        if len(occ) != M or sum(occ) != N or any(o < 0 or o >= d for o in occ):
            raise ValueError("occupations must have length M, lie in [0,d) and sum to N")
        st = cls(M, d, N, chi)
        c = N
        for k in range(M + 1):
            st.sectors[k] = [c]
            st.lam[k] = {c: np.ones(1)}
            if k < M:
                st.gam[k] = {(c, c - occ[k]): np.ones((1, 1), dtype=np.complex128)}
                c -= occ[k]
        return st

    def n(self, k: int, c: int) -> int:
        return len(self.lam[k][c]) if c in self.lam[k] else 0

    def bond_dim(self, k: int) -> int:
        return sum(len(v) for v in self.lam[k].values())

    def copy(self) -> "U1MPS":
        st = U1MPS(self.M, self.d, self.N, self.chi)
        st.sectors = [list(s) for s in self.sectors]
        st.lam = [{c: v.copy() for c, v in l.items()} for l in self.lam]
        st.gam = [{b: v.copy() for b, v in g.items()} for g in self.gam]
        st.log_norm = self.log_norm
        st.discarded_total = self.discarded_total
        return st

    # ---------------------------------------------------------------- the two-site update
    def apply_gate(self, s: int, U: np.ndarray, chi: int | None = None, cutoff: float = 1e-12,
                   record: bool = False) -> GateRecord | None:
        """Charge-blocked two-site update on sites (s, s+1); bonds L=s, C=s+1 (rebuilt), R=s+2.

        U[(out_s*d + out_{s+1}), (in_s*d + in_{s+1})]  (reading S3).  U need not be unitary (S13).
        """
        d, N = self.d, self.N
        chi = self.chi if chi is None else chi
        if not (0 <= s <= self.M - 2):
            raise ValueError("site out of range")
        U = np.asarray(U, dtype=np.complex128).reshape(d * d, d * d)
        L, C, R = s, s + 1, s + 2
        lamL, lamC, lamR = self.lam[L], self.lam[C], self.lam[R]
        gamA, gamB = self.gam[s], self.gam[s + 1]
        rec = GateRecord(site=s)

        # -- step 1 (a1+a2): Theta(c) blocks, Eq.16.  For every (c_l, c_r) and
        #    every NEW centre charge c allowed by the occupations (reading S5), sum over the OLD
        #    centre sectors c' (= the alpha_k sum restricted by the first two deltas of Eq.16).
        blocks: Dict[int, Dict[Block, np.ndarray]] = {}
        for cl in self.sectors[L]:
            for cr in self.sectors[R]:
                if not (0 <= cl - cr <= 2 * (d - 1)):
                    continue
                T = {}
                for cp in self.sectors[C]:
                    jk, jk1 = cl - cp, cp - cr            # input occupations (j_k, j_{k+1})
                    if not (0 <= jk <= d - 1 and 0 <= jk1 <= d - 1):
                        continue
                    if (cl, cp) not in gamA or (cp, cr) not in gamB:
                        continue                          # missing blocks are zero
                    T[cp] = ((lamL[cl][:, None] * gamA[(cl, cp)] * lamC[cp][None, :])
                             @ (gamB[(cp, cr)] * lamR[cr][None, :]))
                for c in range(max(0, cr), min(N, cl) + 1):
                    ik, ik1 = cl - c, c - cr              # output occupations (i_k, i_{k+1})
                    if not (0 <= ik <= d - 1 and 0 <= ik1 <= d - 1):
                        continue
                    blk = np.zeros((len(lamL[cl]), len(lamR[cr])), dtype=np.complex128)
                    for cp, Tcp in T.items():
                        blk = blk + U[ik * d + ik1, (cl - cp) * d + (cp - cr)] * Tcp
                    blocks.setdefault(c, {})[(cl, cr)] = blk

        # -- step 2 (a3): assemble Theta(c) (row blocks ascending c_l, column blocks ascending c_r)
        #    and one thin LAPACK SVD per centre charge (Eq.12 restricted to the sector).
        pool = []
        Vs, Ss, Ws, rowmap, colmap = {}, {}, {}, {}, {}
        for c in sorted(blocks):
            cls_ = sorted({b[0] for b in blocks[c]})
            crs_ = sorted({b[1] for b in blocks[c]})
            roff, off = {}, 0
            for cl in cls_:
                roff[cl] = off
                off += len(lamL[cl])
            nrow = off
            coff, off = {}, 0
            for cr in crs_:
                coff[cr] = off
                off += len(lamR[cr])
            ncol = off
            theta = np.zeros((nrow, ncol), dtype=np.complex128)
            for (cl, cr), blk in blocks[c].items():
                theta[roff[cl]:roff[cl] + blk.shape[0], coff[cr]:coff[cr] + blk.shape[1]] = blk
            V, S, W = np.linalg.svd(theta, full_matrices=False)
            Vs[c], Ss[c], Ws[c] = V, S, W
            rowmap[c] = [(cl, roff[cl], len(lamL[cl])) for cl in cls_]
            colmap[c] = [(cr, coff[cr], len(lamR[cr])) for cr in crs_]
            for j, sv in enumerate(S):
                pool.append((float(sv), c, j))
            if record:
                rec.theta[c] = theta
        if record:
            rec.charges = sorted(blocks)
            rec.rows, rec.cols = rowmap, colmap
            rec.V, rec.sigma, rec.W = Vs, Ss, Ws

        # -- step 3 (a4): global top-chi over all sectors (L121); absolute cutoff first (S7);
        #    order (sigma desc, c asc, j asc) (S8); keep at least one.
        weight_all = sum(p[0] ** 2 for p in pool)
        order = sorted(pool, key=lambda p: (-p[0], p[1], p[2]))
        cand = [p for p in order if p[0] > cutoff]
        kept = cand[:chi]
        if not kept:
            kept = order[:1]
        keep: Dict[int, int] = {}
        for sv, c, j in kept:
            keep[c] = keep.get(c, 0) + 1
        # -- step 4: renormalise (S9)
        w = sum(p[0] ** 2 for p in kept)
        self.log_norm += 0.5 * math.log(w)
        self.discarded_total += weight_all - w
        rec.keep = {c: keep.get(c, 0) for c in sorted(blocks)}
        rec.weight_kept, rec.weight_all, rec.discarded = w, weight_all, weight_all - w
        rec.sigma_chi = kept[-1][0]
        rec.sigma_next = cand[len(kept)][0] if len(cand) > len(kept) else 0.0
        rec.cutoff_gap = min((abs(p[0] - cutoff) for p in pool), default=math.inf)

        # -- step 5 (a5): new bond C and the two Gammas, Eq.13/14 (L96-102, reading S4)
        newA: Dict[Block, np.ndarray] = {}
        newB: Dict[Block, np.ndarray] = {}
        self.sectors[C] = sorted(keep)
        self.lam[C] = {}
        for c in self.sectors[C]:
            kc = keep[c]
            self.lam[C][c] = Ss[c][:kc] / math.sqrt(w)
            for cl, off, nrows in rowmap[c]:
                newA[(cl, c)] = Vs[c][off:off + nrows, :kc] / lamL[cl][:, None]
            for cr, off, ncols in colmap[c]:
                newB[(c, cr)] = Ws[c][:kc, off:off + ncols] / lamR[cr][None, :]
        self.gam[s], self.gam[s + 1] = newA, newB
        return rec if record else None

    # ---------------------------------------------------------------- readouts (a6)
    def norm2(self) -> float:
        return math.exp(2.0 * self.log_norm)

    def expect_n(self, s: int) -> float:
        """Canonical-form <n_s> = sum (c_l-c_r) lam_L^2 |Gamma|^2 lam_R^2 (SURVEY §8(c) Readouts)."""
        tot = 0.0
        for (cl, cr), g in self.gam[s].items():
            wl = self.lam[s][cl] ** 2
            wr = self.lam[s + 1][cr] ** 2
            tot += (cl - cr) * float(wl @ (np.abs(g) ** 2) @ wr)
        return tot

    def bond_entropy(self, k: int) -> float:
        """S_k = -sum lambda^2 ln lambda^2 (natural log, reading S23)."""
        tot = 0.0
        for c in self.sectors[k]:
            p = self.lam[k][c] ** 2
            p = p[p > 0]
            tot -= float(np.sum(p * np.log(p)))
        return tot

    # ---------------------------------------------------------------- oracle-only validators
    def amplitudes(self) -> np.ndarray:
        """Full state vector of length d^M (site 0 = most significant digit, S23); Eq.15 written out."""
        M, d = self.M, self.d
        # cur[c] : (d^s, n_s(c)) partial amplitudes including lambda of the bond on their right
        cur = {self.N: np.ones((1, 1), dtype=np.complex128)}
        for s in range(M):
            nxt: Dict[int, np.ndarray] = {}
            rows = d ** s
            for cr in self.sectors[s + 1]:
                acc = np.zeros((rows * d, len(self.lam[s + 1][cr])), dtype=np.complex128)
                hit = False
                for i in range(d):
                    cl = cr + i
                    if cl in cur and (cl, cr) in self.gam[s]:
                        acc[i::d, :] = cur[cl] @ self.gam[s][(cl, cr)]
                        hit = True
                if hit:
                    nxt[cr] = acc * self.lam[s + 1][cr][None, :]
            cur = nxt
        return cur[0][:, 0] if 0 in cur else np.zeros(d ** M, dtype=np.complex128)

    def expect_n_full(self, s: int) -> float:
        """<psi|n_s|psi>/<psi|psi> with explicitly contracted left and right environments (pin P10)."""
        # left environments E_k[c] (n_k(c) x n_k(c)) for the tensors A^[s] = Gamma^[s] lambda^[s+1]
        def A(site, cl, cr):
            return self.gam[site][(cl, cr)] * self.lam[site + 1][cr][None, :]
        E = {self.N: np.ones((1, 1), dtype=np.complex128)}
        envL = [E]
        for site in range(self.M):
            En: Dict[int, np.ndarray] = {}
            for (cl, cr) in self.gam[site]:
                if cl in E:
                    a = A(site, cl, cr)
                    En[cr] = En.get(cr, 0) + a.conj().T @ E[cl] @ a
            E = En
            envL.append(E)
        norm = float(np.real(envL[self.M][0][0, 0]))
        Rr = {0: np.ones((1, 1), dtype=np.complex128)}
        for site in range(self.M - 1, s, -1):
            Rn: Dict[int, np.ndarray] = {}
            for (cl, cr) in self.gam[site]:
                if cr in Rr:
                    a = A(site, cl, cr)
                    Rn[cl] = Rn.get(cl, 0) + a @ Rr[cr] @ a.conj().T
            Rr = Rn
        val = 0.0
        for (cl, cr) in self.gam[s]:
            if cl in envL[s] and cr in Rr:
                a = A(s, cl, cr)
                val += (cl - cr) * float(np.real(np.trace(a.conj().T @ envL[s][cl] @ a @ Rr[cr])))
        return val / norm

    def expect_nn_full(self, j: int, k: int) -> float:
        """<psi|n_j n_k|psi>/<psi|psi>, j <= k, with explicitly contracted environments (pin P12).

        Same contraction as expect_n_full (state of Eq.15): the occupation of a site is the charge
        difference of its two bonds, so n_j inserts the weight (c_l - c_r) into the transfer step of site j.
        """
        if j > k:
            j, k = k, j

        def A(site, cl, cr):
            return self.gam[site][(cl, cr)] * self.lam[site + 1][cr][None, :]
        E = {self.N: np.ones((1, 1), dtype=np.complex128)}
        F = None                                   # left environment with n_j inserted, from bond j+1 on
        for site in range(k):
            En: Dict[int, np.ndarray] = {}
            Fn: Dict[int, np.ndarray] = {}
            for (cl, cr) in self.gam[site]:
                a = A(site, cl, cr)
                if cl in E:
                    En[cr] = En.get(cr, 0) + a.conj().T @ E[cl] @ a
                    if site == j:
                        Fn[cr] = Fn.get(cr, 0) + (cl - cr) * (a.conj().T @ E[cl] @ a)
                if F is not None and cl in F:
                    Fn[cr] = Fn.get(cr, 0) + a.conj().T @ F[cl] @ a
            E = En
            if site >= j:
                F = Fn
        Rr = {0: np.ones((1, 1), dtype=np.complex128)}
        for site in range(self.M - 1, k, -1):
            Rn: Dict[int, np.ndarray] = {}
            for (cl, cr) in self.gam[site]:
                if cr in Rr:
                    a = A(site, cl, cr)
                    Rn[cl] = Rn.get(cl, 0) + a @ Rr[cr] @ a.conj().T
            Rr = Rn
        val, norm = 0.0, 0.0
        for (cl, cr) in self.gam[k]:
            if cr not in Rr:
                continue
            a = A(k, cl, cr)
            if cl in E:
                t = float(np.real(np.trace(a.conj().T @ E[cl] @ a @ Rr[cr])))
                norm += t
                if j == k:
                    val += (cl - cr) ** 2 * t
            if j < k and F is not None and cl in F:
                val += (cl - cr) * float(np.real(np.trace(a.conj().T @ F[cl] @ a @ Rr[cr])))
        return val / norm

    def sample_fock(self, u: np.ndarray):
        """Fock patterns (n_0 .. n_{M-1}) drawn from |<n|psi>|^2 / <psi|psi>, site by site (pin P13).

        The use the boson-sampling section motivates (Eq.7-8: the output distribution over occupation
        patterns), on the state of Eq.15 (L112-114: the occupation of a site is the charge difference of its bonds).
        The uniform numbers are an INPUT: u[b, s] in [0, 1) decides site s of sample b by inverse CDF over the
        occupations in ascending order.  With A^[s](cl, cr) = Gamma^[s][cl, cr] diag(lambda^[s+1][cr]) and the right
        environments R_M = {0: [[1]]}, R_s[cl] = sum_cr A R_{s+1}[cr] A^H (as in expect_n_full), a sample that has
        reached bond s with charge c and boundary row vector v (v = [1] at bond 0) takes occupation i with weight
            p_i = w_i R_{s+1}[c - i] w_i^H,   w_i = v A^[s](c, c - i),
        chosen as the smallest i with u * sum_i' p_i' < p_0 + .. + p_i; then v <- w_i / sqrt(p_i), c <- c - i.
        Exact for whatever Gamma, lambda the state holds (no canonical form assumed).

        Returns (pattern int64 [B, M], logp float64 [B] = ln of the probability of the drawn pattern, margin float64
        [B] = the smallest distance of u * sum p from a CDF step that was compared, relative to sum p: a draw with a
        tiny margin is decided by rounding and is not comparable between implementations).
        """
        u = np.asarray(u, dtype=np.float64)
        B, M = u.shape
        assert M == self.M

        def A(site, cl, cr):
            return self.gam[site][(cl, cr)] * self.lam[site + 1][cr][None, :]
        R = [None] * (M + 1)
        R[M] = {0: np.ones((1, 1), dtype=np.complex128)}
        for site in range(M - 1, -1, -1):
            Rn: Dict[int, np.ndarray] = {}
            for (cl, cr) in self.gam[site]:
                if cr in R[site + 1]:
                    a = A(site, cl, cr)
                    Rn[cl] = Rn.get(cl, 0) + a @ R[site + 1][cr] @ a.conj().T
            R[site] = Rn
        pattern = np.zeros((B, M), dtype=np.int64)
        logp = np.zeros(B)
        margin = np.full(B, np.inf)
        for b in range(B):
            v = np.ones(1, dtype=np.complex128)
            c = self.N
            for site in range(M):
                w = [None] * self.d
                p = np.zeros(self.d)
                for i in range(self.d):
                    cr = c - i
                    if (c, cr) in self.gam[site] and cr in R[site + 1]:
                        w[i] = v @ A(site, c, cr)
                        p[i] = float(np.real(w[i] @ R[site + 1][cr] @ w[i].conj()))
                tot = 0.0
                for i in range(self.d):
                    tot += p[i]
                target = u[b, site] * tot
                cum, pick = 0.0, -1
                for i in range(self.d):
                    cum += p[i]
                    if p[i] > 0.0:
                        if pick < 0:
                            margin[b] = min(margin[b], abs(target - cum) / tot)
                        if pick < 0 and target < cum:
                            pick = i
                if pick < 0:                      # rounding at the top of the CDF: the last occupation with weight
                    pick = max(i for i in range(self.d) if p[i] > 0.0)
                pattern[b, site] = pick
                logp[b] += math.log(p[pick] / tot)
                v = w[pick] / math.sqrt(p[pick])
                c -= pick
        return pattern, logp, margin

    def to_dense(self):
        """Expand to a plain (non-symmetric) Vidal MPS: Gamma^[s]i (d, D_s, D_{s+1}), lambda^[k] (pin P6)."""
        offs = []
        for k in range(self.M + 1):
            o, off = {}, 0
            for c in self.sectors[k]:
                o[c] = off
                off += len(self.lam[k][c])
            offs.append((o, off))
        lams = [np.concatenate([self.lam[k][c] for c in self.sectors[k]]) for k in range(self.M + 1)]
        gams = []
        for s in range(self.M):
            g = np.zeros((self.d, offs[s][1], offs[s + 1][1]), dtype=np.complex128)
            for (cl, cr), blk in self.gam[s].items():
                i = cl - cr
                g[i, offs[s][0][cl]:offs[s][0][cl] + blk.shape[0],
                  offs[s + 1][0][cr]:offs[s + 1][0][cr] + blk.shape[1]] = blk
            gams.append(g)
        return gams, lams


def dense_two_site_sigma(gams, lams, s: int, U: np.ndarray, d: int) -> np.ndarray:
    """Singular values of the plain d*chi x d*chi Theta of Eq.11-12: brute force for P6."""
    U4 = np.asarray(U, dtype=np.complex128).reshape(d, d, d, d)      # [out_a, out_b, in_a, in_b]
    A = lams[s][None, :, None] * gams[s] * lams[s + 1][None, None, :]       # i, a, b
    B = gams[s + 1] * lams[s + 2][None, None, :]                              # j, b, g
    theta = np.einsum("xyij,iab,jbg->xayg", U4, A, B)
    Dl, Dr = theta.shape[1], theta.shape[3]
    return np.linalg.svd(theta.reshape(d * Dl, d * Dr), compute_uv=False)


def run_columns(st: U1MPS, columns, chi=None, cutoff=1e-12):
    """Apply gate columns [(sites, U[g])...] in order (a brick-wall layer = two columns, reading S15)."""
    for sites, us in columns:
        for g, s in enumerate(sites):
            st.apply_gate(int(s), us[g], chi=chi, cutoff=cutoff)
    return st
