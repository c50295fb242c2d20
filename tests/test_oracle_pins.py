"""Pins P1-P10 of SURVEY.md §8(c): the oracle against what the paper and the mathematics fix.

None of these re-type the oracle's formulae: they compare against an exact d^M state vector
(tests/statevector_ref.py), a brute-force dense (non-symmetric) SVD, permanents, single-particle
propagation and library routines (scipy expm / numpy svd).
"""
import itertools
import math

import numpy as np
import pytest
import scipy.linalg

import statevector_ref as sv
from paper_2303_11409_b200 import inputs
from u1mps_oracle import U1MPS, dense_two_site_sigma, run_columns


def evolve_both(M, d, N, occ, gates, chi, cutoff=1e-12):
    st = U1MPS.product_state(M, d, N, chi, occ)
    vec = sv.product_vector(occ, d)
    for s, U in gates:
        st.apply_gate(s, U, cutoff=cutoff)
        vec = sv.apply_two_site(vec, M, d, s, U)
    return st, vec


def brick_gates(rng, M, d, layers, gen):
    out = []
    for t in range(2 * layers):
        for s in inputs.column_sites(M, t):
            out.append((s, gen(rng)))
    return out


# ------------------------------------------------------------------ gate generators (inputs.py)
def test_xxz_gate_matches_expm():
    sx = np.array([[0, 1], [1, 0]], dtype=complex)
    sy = np.array([[0, -1j], [1j, 0]])
    sz = np.diag([1.0, -1.0]).astype(complex)          # index 0 <-> n=0 <-> sz=+1  (Eq.3)
    for delta, dt in [(0.5, 0.05), (1.3, 0.7), (0.0, 0.2)]:
        H = np.kron(sx, sx) + np.kron(sy, sy) + delta * np.kron(sz, sz)
        ref = scipy.linalg.expm(-1j * dt * H)
        assert np.allclose(inputs.xxz_gate(delta, dt), ref, atol=1e-14)


def test_beam_splitter_gate_matches_expm_of_generator():
    rng = np.random.default_rng(5)
    for _ in range(4):
        u = inputs.beam_splitter_2x2(rng.uniform(0, math.pi / 2), rng.uniform(0, 2 * math.pi))
        K = scipy.linalg.logm(u)
        for n in range(0, 6):
            # sector of total photon number n: basis |m, n-m>, m = 0..n; generator sum K[k,j] a_k^+ a_j
            dim = n + 1
            G = np.zeros((dim, dim), dtype=complex)
            for m in range(dim):
                n1, n2 = m, n - m
                G[m, m] += K[0, 0] * n1 + K[1, 1] * n2
                if n2 > 0:   # a_1^+ a_2 |n1,n2> = sqrt((n1+1) n2) |n1+1,n2-1>
                    G[m + 1, m] += K[0, 1] * math.sqrt((n1 + 1) * n2)
                if n1 > 0:   # a_2^+ a_1
                    G[m - 1, m] += K[1, 0] * math.sqrt(n1 * (n2 + 1))
            ref = scipy.linalg.expm(G)
            d = n + 1
            B = inputs.beam_splitter_gate(u, d)
            idx = [m * d + (n - m) for m in range(dim)]
            assert np.allclose(B[np.ix_(idx, idx)], ref, atol=1e-12)
            assert np.allclose(ref.conj().T @ ref, np.eye(dim), atol=1e-12)


def test_gates_conserve_charge_and_haar_unitary():
    rng = np.random.default_rng(1)
    for d, g in [(2, inputs.hardcore_haar_gate(rng)), (4, inputs.haar_beam_splitter_gate(rng, 4)),
                 (3, inputs.random_u1_gate(rng, 3)), (2, inputs.xxz_gate(0.5, 0.05))]:
        for r, c in itertools.product(range(d * d), repeat=2):
            if (r // d + r % d) != (c // d + c % d):
                assert g[r, c] == 0
    u = inputs.hardcore_haar_gate(rng)
    assert np.allclose(u.conj().T @ u, np.eye(4), atol=1e-14)


def test_workload_gate_counts():
    assert inputs.WORKLOADS[1].n_gates == 15
    assert inputs.WORKLOADS[2].n_gates == 1260
    assert inputs.WORKLOADS[3].n_gates == 6350
    assert inputs.WORKLOADS[4].n_gates == 496
    assert inputs.WORKLOADS[5].n_gates == 4950


# ------------------------------------------------------------------ P1: exact state vector
def test_P1_config1_exact_statevector():
    """BASELINE.json config 1: M=16, N=8, chi=32, one brick-wall layer; all 2^16 amplitudes (Eq.9)."""
    w = inputs.WORKLOADS[1]
    st = U1MPS.product_state(w.M, w.d, w.N, w.chi, w.occ)
    vec = sv.product_vector(w.occ, w.d)
    ng = 0
    for sites, us in inputs.gate_columns(w):
        for g, s in enumerate(sites):
            st.apply_gate(int(s), us[g], cutoff=w.cutoff)
            vec = sv.apply_two_site(vec, w.M, w.d, int(s), us[g])
            ng += 1
    assert ng == 15
    amp = st.amplitudes()
    assert np.max(np.abs(amp - vec)) < 1e-12
    assert max(st.bond_dim(k) for k in range(w.M + 1)) <= 4          # no truncation is triggered
    assert abs(st.norm2() - 1.0) < 1e-12


@pytest.mark.parametrize("d,M,N,layers,seed", [(2, 10, 5, 5, 0), (3, 7, 6, 3, 1), (4, 6, 7, 3, 2), (5, 5, 6, 2, 3)])
def test_P1_random_generic_u1_gates(d, M, N, layers, seed):
    """Generic (non-symmetric-looking) random U(1) unitaries: pins U's index roles (S3), Eq.16's deltas, Eq.13/14."""
    rng = np.random.default_rng(seed)
    occ = [0] * M
    left = N
    for s in range(M):
        occ[s] = min(d - 1, left)
        left -= occ[s]
    occ = list(rng.permutation(occ))
    gates = brick_gates(rng, M, d, layers, lambda r: inputs.random_u1_gate(r, d))
    st, vec = evolve_both(M, d, N, occ, gates, chi=d ** (M // 2))
    assert np.max(np.abs(st.amplitudes() - vec)) < 1e-12
    assert abs(st.norm2() - 1.0) < 1e-12


def test_P1_nonunitary_gates_keep_the_state_exact():
    """S13: U need not be unitary; amplitudes * sqrt(norm2) follow the raw state vector."""
    rng = np.random.default_rng(7)
    d, M, N = 3, 6, 5
    occ = [2, 0, 1, 1, 0, 1]
    gates = brick_gates(rng, M, d, 2, lambda r: inputs.random_u1_gate(r, d, unitary=False))
    st, vec = evolve_both(M, d, N, occ, gates, chi=d ** 3, cutoff=0.0)
    amp = st.amplitudes() * math.sqrt(st.norm2())
    assert np.max(np.abs(amp - vec)) < 1e-11 * np.max(np.abs(vec))


# ------------------------------------------------------------------ P2/P3/P4: invariants
def _random_state(d, M, N, chi, layers, seed, gen=None):
    rng = np.random.default_rng(seed)
    occ = [0] * M
    left = N
    for s in range(0, M, 2):
        occ[s] = min(d - 1, left)
        left -= occ[s]
    for s in range(1, M, 2):
        occ[s] = min(d - 1, left)
        left -= occ[s]
    assert left == 0
    st = U1MPS.product_state(M, d, N, chi, occ)
    gen = gen or (lambda r: inputs.random_u1_gate(r, d))
    for s, U in brick_gates(rng, M, d, layers, gen):
        st.apply_gate(s, U)
    return st


def test_P2_charge_structure_and_total_number():
    st = _random_state(3, 10, 9, 243, 4, 11)
    assert st.sectors[0] == [st.N] and st.sectors[st.M] == [0]
    for s in range(st.M):
        for (cl, cr), blk in st.gam[s].items():
            assert 0 <= cl - cr <= st.d - 1
            assert blk.shape == (st.n(s, cl), st.n(s + 1, cr))
    for k in range(st.M + 1):
        assert st.sectors[k] == sorted(st.sectors[k])
        for c in st.sectors[k]:
            lam = st.lam[k][c]
            assert np.all(lam > 0) and np.all(np.diff(lam) <= 0)
    assert abs(sum(st.expect_n(s) for s in range(st.M)) - st.N) < 1e-12


def test_P3_unit_norm_before_renormalising():
    """Unitary U, no truncation => sum sigma^2 = 1 at every gate (canonical environments are orthonormal)."""
    rng = np.random.default_rng(3)
    d, M, N = 2, 12, 6
    st = U1MPS.product_state(M, d, N, 64, [1, 0] * 6)
    for s, U in brick_gates(rng, M, d, 6, inputs.hardcore_haar_gate):
        rec = st.apply_gate(s, U, record=True)
        assert abs(rec.weight_all - 1.0) < 1e-13
        assert rec.discarded < 1e-20


def test_P4_canonical_form_identities():
    st = _random_state(3, 8, 7, 81, 3, 5)
    for s in range(st.M):
        # left:  sum_{c_l} Gamma^+ lam_L^2 Gamma = 1 per right sector;  right: Gamma lam_R^2 Gamma^+ = 1
        left, right = {}, {}
        for (cl, cr), g in st.gam[s].items():
            left[cr] = left.get(cr, 0) + g.conj().T @ (st.lam[s][cl][:, None] ** 2 * g)
            right[cl] = right.get(cl, 0) + (g * st.lam[s + 1][cr][None, :] ** 2) @ g.conj().T
        for c, m in left.items():
            assert np.allclose(m, np.eye(m.shape[0]), atol=1e-12)
        for c, m in right.items():
            assert np.allclose(m, np.eye(m.shape[0]), atol=1e-12)
    for k in range(st.M + 1):
        assert abs(sum(float(np.sum(v ** 2)) for v in st.lam[k].values()) - 1.0) < 1e-12


# ------------------------------------------------------------------ P5/P6: SVD and truncation
def test_P5_eckart_young_per_sector():
    st = _random_state(2, 12, 6, 64, 6, 9, gen=inputs.hardcore_haar_gate)
    rng = np.random.default_rng(10)
    before = st.copy()
    rec = st.apply_gate(5, inputs.hardcore_haar_gate(rng), chi=6, record=True)
    assert sum(rec.keep.values()) == 6
    for c in rec.charges:
        k = rec.keep[c]
        approx = (rec.V[c][:, :k] * rec.sigma[c][:k][None, :]) @ rec.W[c][:k, :]
        err = np.linalg.norm(rec.theta[c] - approx) ** 2
        assert abs(err - float(np.sum(rec.sigma[c][k:] ** 2))) < 1e-13
        full = (rec.V[c] * rec.sigma[c][None, :]) @ rec.W[c]
        assert np.linalg.norm(rec.theta[c] - full) < 1e-13
    assert abs(rec.discarded - (rec.weight_all - rec.weight_kept)) < 1e-15
    # new tensors are V / lambda_L and W / lambda_R (Eq.13/14)
    for c in st.sectors[6]:
        for cl, off, nrows in rec.rows[c]:
            assert np.allclose(before.lam[5][cl][:, None] * st.gam[5][(cl, c)], rec.V[c][off:off + nrows, :rec.keep[c]])
        for cr, off, ncols in rec.cols[c]:
            assert np.allclose(st.gam[6][(c, cr)] * before.lam[7][cr][None, :], rec.W[c][:rec.keep[c], off:off + ncols])


@pytest.mark.parametrize("d,M,N,seed", [(2, 10, 5, 21), (3, 8, 8, 22), (4, 6, 9, 23)])
def test_P6_brute_force_dense_svd(d, M, N, seed):
    """Union of per-sector sigma == non-zero sigma of the plain d*chi x d*chi Theta (PAPER.md L89-94 vs L116-123)."""
    st = _random_state(d, M, N, 256, 3, seed)
    rng = np.random.default_rng(seed + 100)
    for s in [0, M // 2 - 1, M // 2, M - 2]:
        U = inputs.random_u1_gate(rng, d)
        gams, lams = st.to_dense()
        dense = dense_two_site_sigma(gams, lams, s, U, d)
        chi_cut = max(2, st.bond_dim(s + 1) // 2)
        rec = st.copy().apply_gate(s, U, chi=chi_cut, record=True)
        sym = np.sort(np.concatenate([rec.sigma[c] for c in rec.charges]))[::-1]
        nz = dense[dense > 1e-13]
        assert len(sym[sym > 1e-13]) == len(nz)
        assert np.max(np.abs(sym[:len(nz)] - nz)) < 1e-13
        kept = np.sort(np.concatenate([rec.sigma[c][:rec.keep[c]] for c in rec.charges]))[::-1]
        assert len(kept) == min(chi_cut, len(nz))
        assert np.max(np.abs(kept - dense[:len(kept)])) < 1e-13       # the global top-chi (L121)


# ------------------------------------------------------------------ P7: identity / swap
def test_P7_identity_gate_is_a_fixed_point():
    st = _random_state(3, 8, 7, 81, 3, 31)
    amp0 = st.amplitudes()
    lam0 = [{c: v.copy() for c, v in l.items()} for l in st.lam]
    for s in range(st.M - 1):
        st.apply_gate(s, np.eye(9))
    assert np.max(np.abs(st.amplitudes() - amp0)) < 1e-12
    for k in range(st.M + 1):
        assert set(st.lam[k]) == set(lam0[k])
        for c in lam0[k]:
            assert np.allclose(st.lam[k][c], lam0[k][c], atol=1e-13)


def test_P7_swap_permutes_a_product_state():
    d, occ = 4, [3, 0, 2, 1, 0]
    st = U1MPS.product_state(5, d, 6, 8, occ)
    st.apply_gate(1, inputs.swap_gate(d))
    st.apply_gate(2, inputs.swap_gate(d))
    want = [3, 2, 1, 0, 0]
    vec = st.amplitudes()
    ref = sv.product_vector(want, d)
    assert np.max(np.abs(np.abs(vec) - np.abs(ref))) < 1e-14
    assert [round(st.expect_n(s)) for s in range(5)] == want
    assert all(st.bond_dim(k) == 1 for k in range(6))


# ------------------------------------------------------------------ P8: closed forms
def test_P8_single_particle_walk():
    """N=1: amplitudes are a column of the product of the embedded 2x2 mode unitaries."""
    rng = np.random.default_rng(41)
    M, d = 9, 2
    occ = [0] * M
    occ[4] = 1
    st = U1MPS.product_state(M, d, 1, 4, occ)
    W = np.eye(M, dtype=complex)
    for t in range(6):
        for s in inputs.column_sites(M, t):
            u = inputs.beam_splitter_2x2(rng.uniform(0, math.pi / 2), rng.uniform(0, 2 * math.pi))
            st.apply_gate(s, inputs.beam_splitter_gate(u, d))
            E = np.eye(M, dtype=complex)
            E[s:s + 2, s:s + 2] = u
            W = E @ W
    amp = st.amplitudes()
    for k in range(M):
        idx = d ** (M - 1 - k)
        assert abs(amp[idx] - W[k, 4]) < 1e-13
    assert all(st.bond_dim(k) <= 2 for k in range(M + 1))


def test_P8_hong_ou_mandel():
    u = inputs.beam_splitter_2x2(math.pi / 4, 0.3)
    st = U1MPS.product_state(2, 3, 2, 9, [1, 1])
    st.apply_gate(0, inputs.beam_splitter_gate(u, 3))
    amp = st.amplitudes().reshape(3, 3)
    assert abs(amp[1, 1]) < 1e-15
    assert abs(abs(amp[2, 0]) ** 2 - 0.5) < 1e-14 and abs(abs(amp[0, 2]) ** 2 - 0.5) < 1e-14


def test_P8_permanents_of_the_mesh_unitary():
    """d > N so nothing is cut off: Fock amplitudes = permanents of sub-matrices (Eq.8)."""
    rng = np.random.default_rng(43)
    M, N = 5, 3
    d = N + 1
    occ = [1, 1, 1, 0, 0]
    st = U1MPS.product_state(M, d, N, 64, occ)
    Um = np.eye(M, dtype=complex)
    for t in range(M):
        for s in inputs.column_sites(M, t):
            u = inputs.beam_splitter_2x2(math.acos(math.sqrt(rng.uniform())), rng.uniform(0, 2 * math.pi))
            st.apply_gate(s, inputs.beam_splitter_gate(u, d))
            E = np.eye(M, dtype=complex)
            E[s:s + 2, s:s + 2] = u
            Um = E @ Um
    amp = st.amplitudes()
    checked = 0
    for m_out in itertools.product(range(d), repeat=M):
        if sum(m_out) != N:
            continue
        idx = 0
        for m in m_out:
            idx = idx * d + m
        assert abs(amp[idx] - sv.fock_amplitude(Um, occ, m_out)) < 1e-12
        checked += 1
    assert checked == math.comb(N + M - 1, M - 1)


# ------------------------------------------------------------------ P9: free case
def test_P9_free_fermion_densities():
    """XXZ gate at Delta=0 (XX chain == free fermions): <n_k> from the M x M correlation matrix (Eq.3-4)."""
    M, N, dt, layers = 20, 10, 0.05, 10
    occ = [s % 2 for s in range(M)]
    st = U1MPS.product_state(M, 2, N, 128, occ)
    U = inputs.xxz_gate(0.0, dt)
    C = np.diag(np.asarray(occ, dtype=complex))            # C_ij = <f_i^+ f_j>
    w2 = U[1:3, 1:3][::-1, ::-1]                            # block on (|10>,|01>) = sites (s, s+1) occupied
    for t in range(2 * layers):
        for s in inputs.column_sites(M, t):
            st.apply_gate(s, U)
            Wm = np.eye(M, dtype=complex)
            Wm[s:s + 2, s:s + 2] = w2
            C = Wm.conj() @ C @ Wm.T
    dens = np.real(np.diag(C))
    got = np.array([st.expect_n(s) for s in range(M)])
    assert st.discarded_total < 1e-18
    assert np.max(np.abs(got - dens)) < 1e-10


# ------------------------------------------------------------------ P10: readout formula
def test_P10_readouts_match_state_vector_and_environments():
    rng = np.random.default_rng(51)
    d, M, N = 3, 7, 6
    occ = [2, 0, 1, 1, 0, 2, 0]
    gates = brick_gates(rng, M, d, 3, lambda r: inputs.random_u1_gate(r, d))
    st, vec = evolve_both(M, d, N, occ, gates, chi=d ** 3)
    for s in range(M):
        ref = sv.number_expectation(vec, M, d, s)
        assert abs(st.expect_n(s) - ref) < 1e-12
        assert abs(st.expect_n_full(s) - ref) < 1e-12
    for k in range(1, M):
        p = sv.schmidt_values(vec, M, d, k) ** 2
        p = p[p > 1e-30]
        assert abs(st.bond_entropy(k) - float(-np.sum(p * np.log(p)))) < 1e-11
        lam = np.sort(np.concatenate([st.lam[k][c] for c in st.sectors[k]]))[::-1]
        assert np.max(np.abs(lam - sv.schmidt_values(vec, M, d, k)[:len(lam)])) < 1e-12
    assert set(sv.total_charge_weights(vec, M, d)) == {N}


def test_truncation_is_reported_and_state_stays_normalised():
    """Config-2 family at reduced size: truncation at chi with global ordering across sectors."""
    w = inputs.small_variant(inputs.WORKLOADS[2], M=14, N=7, chi=16, columns=8)
    st = U1MPS.product_state(w.M, w.d, w.N, w.chi, w.occ)
    vec = sv.product_vector(w.occ, w.d)
    for sites, us in inputs.gate_columns(w):
        for g, s in enumerate(sites):
            st.apply_gate(int(s), us[g], cutoff=w.cutoff)
            vec = sv.apply_two_site(vec, w.M, w.d, int(s), us[g])
    assert max(st.bond_dim(k) for k in range(w.M + 1)) == 16
    assert st.discarded_total > 1e-6
    amp = st.amplitudes()
    fid = abs(np.vdot(vec, amp)) ** 2 / float(np.vdot(amp, amp).real)
    assert 0.5 < fid < 1.0 - 1e-9                         # approximate, but close
    # canonical-form <n> is only approximate once truncation has broken canonicity (SURVEY §8(c) Readouts)
    assert abs(sum(st.expect_n(s) for s in range(w.M)) - w.N) < 2e-2
    assert abs(sum(st.expect_n_full(s) for s in range(w.M)) - w.N) < 1e-11


# ------------------------------------------------------------------ P11: the order at the cut (readings S7, S8)
def test_P11_tie_order_and_keep_at_least_one():
    """DESIGN reading S8 (the paper is silent): ties at the chi-th value go to (sigma desc, c asc, j asc); reading S7:
    at least one value is always kept.  Constructed exact ties: the hop / stay gate below splits |..10..> into two
    charge sectors with bitwise equal singular values.  The expected kept set is worked out here from the dense Theta of
    Eq.11 (one plain SVD per charge block cut out of the dense matrix by the occupations - not by the oracle's sector
    code) with the rule written out again; a c-descending or j-descending tie-break fails."""
    a = 0.7071067811865476
    U = np.zeros((4, 4), dtype=np.complex128)
    U[0, 0] = U[3, 3] = 1.0
    U[1, 1] = U[1, 2] = U[2, 1] = a
    U[2, 2] = -a
    # two-site chain: Theta(c = 0) = [a], Theta(c = 1) = [a]
    st = U1MPS.product_state(2, 2, 1, 4, [1, 0])
    rec = st.apply_gate(0, U, chi=1, cutoff=1e-12, record=True)
    assert rec.sigma[0][0] == rec.sigma[1][0] == a          # an exact tie
    assert rec.keep == {0: 1, 1: 0} and st.sectors[1] == [0]
    # keep at least one: a cutoff above every singular value keeps the first of the order, nothing else
    st = U1MPS.product_state(2, 2, 1, 4, [1, 0])
    rec = st.apply_gate(0, U, chi=4, cutoff=2.0, record=True)
    assert rec.keep == {0: 1, 1: 0} and abs(st.lam[1][0][0] - 1.0) < 1e-15
    # a chain where the tied sectors hold several values each: two hop / stay gates on |1010> make bond 2 carry the
    # sectors c = 0, 1, 2; the middle gate then sees degenerate pairs across sectors
    st = U1MPS.product_state(4, 2, 2, 16, [1, 0, 1, 0])
    st.apply_gate(0, U, cutoff=1e-12)
    st.apply_gate(2, U, cutoff=1e-12)
    gams, lams = st.to_dense()
    ref = st.copy()
    for chi in (1, 2, 3):
        t = ref.copy()
        rec = t.apply_gate(1, U, chi=chi, cutoff=1e-12, record=True)
        # dense Theta of Eq.11, rows (i, alpha), columns (j, gamma); charge of a column = charge of gamma + j
        U4 = U.reshape(2, 2, 2, 2)
        A = lams[1][None, :, None] * gams[1] * lams[2][None, None, :]
        B = gams[2] * lams[3][None, None, :]
        theta = np.einsum("xyij,iab,jbg->xayg", U4, A, B)
        cR = np.concatenate([[c] * len(st.lam[3][c]) for c in st.sectors[3]])
        pool = []
        for c in range(0, 3):
            cols = [(y, g_) for y in range(2) for g_ in range(len(cR)) if cR[g_] + y == c]
            if not cols:
                continue
            blk = np.stack([theta[:, :, y, g_].reshape(-1) for y, g_ in cols], axis=1)
            sv_ = np.linalg.svd(blk, compute_uv=False)
            pool += [(float(x), c, j) for j, x in enumerate(sv_) if x > 1e-12]
        order = sorted(pool, key=lambda p: (-p[0], p[1], p[2]))[:chi]
        want = {}
        for _, c, _ in order:
            want[c] = want.get(c, 0) + 1
        assert {c: k for c, k in rec.keep.items() if k > 0} == want, (chi, rec.keep, want)
    sig = sorted((float(x), c) for c, v in rec.sigma.items() for x in v if x > 1e-12)
    assert any(abs(x - y) == 0.0 and c1 != c2 for (x, c1), (y, c2) in zip(sig[:-1], sig[1:]))   # ties across sectors exist


# ------------------------------------------------------------------ P12: two-point function with explicit environments
def test_P12_two_point_function_matches_state_vector():
    """<n_j n_k> from the environment contraction against the plain state vector (digit sums over the d^M amplitudes),
    on an untruncated state and on a truncated one (compared with the state vector of the TRUNCATED MPS, rebuilt from
    its amplitudes: the contraction is exact for whatever state the MPS holds)."""
    rng = np.random.default_rng(77)
    d, M, N = 3, 6, 5
    occ = [2, 0, 1, 1, 0, 1]
    gates = brick_gates(rng, M, d, 3, lambda r: inputs.random_u1_gate(r, d))
    for chi in (d ** 3, 4):
        st = U1MPS.product_state(M, d, N, chi, occ)
        for s, U in gates:
            st.apply_gate(s, U, chi=chi, cutoff=1e-12)
        vec = st.amplitudes()
        p = np.abs(vec) ** 2
        p = p / p.sum()
        digits = np.array(list(itertools.product(range(d), repeat=M)))      # site 0 = most significant digit (S23)
        for j in range(M):
            for k in range(j, M):
                ref = float(np.sum(p * digits[:, j] * digits[:, k]))
                assert abs(st.expect_nn_full(j, k) - ref) < 1e-12, (chi, j, k)
        assert abs(sum(st.expect_nn_full(j, k) * (1 if j == k else 2) for j in range(M) for k in range(j, M)) - N * N) < 1e-10


# ------------------------------------------------------------------ P13: Fock-pattern sampling
def _brute_force_sampling(vec, d, M, u):
    """Site-by-site inverse-CDF sampling straight from the d^M amplitudes: the conditional weight of occupation i at site
    s given the prefix is the sum of |amplitude|^2 over all suffixes (site 0 = most significant digit, S23)."""
    P = (np.abs(vec) ** 2).reshape((d,) * M)
    total = P.sum()
    pats, logps, margins = [], [], []
    for b in range(u.shape[0]):
        sub, pat, margin = P, [], np.inf
        for s in range(M):
            w = sub.reshape(d, -1).sum(axis=1)
            target, cum, pick = u[b, s] * w.sum(), 0.0, -1
            for i in range(d):
                cum += w[i]
                if w[i] > 0.0 and pick < 0:
                    margin = min(margin, abs(target - cum) / w.sum())
                    if target < cum:
                        pick = i
            if pick < 0:
                pick = max(i for i in range(d) if w[i] > 0.0)
            pat.append(pick)
            sub = sub[pick]
        pats.append(pat); logps.append(math.log(float(sub) / total)); margins.append(margin)
    return np.array(pats), np.array(logps), np.array(margins)


def test_P13_fock_sampling_matches_conditionals_of_the_state_vector():
    """sample_fock against brute-force conditional sampling over the state vector with the same uniform numbers, on an
    untruncated and on a truncated (non-canonical) state: same patterns, ln P(pattern) = ln(|<n|psi>|^2 / <psi|psi>);
    every drawn pattern conserves the particle number; a product state always returns its own pattern."""
    rng = np.random.default_rng(131)
    d, M, N = 3, 6, 5
    occ = [2, 0, 1, 1, 0, 1]
    gates = brick_gates(rng, M, d, 3, lambda r: inputs.random_u1_gate(r, d))
    u = rng.random((200, M))
    for chi in (d ** 3, 4):
        st = U1MPS.product_state(M, d, N, chi, occ)
        for s, U in gates:
            st.apply_gate(s, U, chi=chi, cutoff=1e-12)
        if chi == 4:
            assert st.discarded_total > 1e-4                      # the truncated state is not canonical any more
        pat, logp, margin = st.sample_fock(u)
        ref_pat, ref_logp, ref_margin = _brute_force_sampling(st.amplitudes(), d, M, u)
        safe = np.minimum(margin, ref_margin) > 1e-9
        assert safe.sum() >= 198
        assert np.array_equal(pat[safe], ref_pat[safe]), chi
        assert np.max(np.abs(logp[safe] - ref_logp[safe])) < 1e-10
        assert np.all(pat.sum(axis=1) == N)
        assert len({tuple(r) for r in pat}) > 20                    # a spread-out distribution, not one pattern
        # the empirical frequencies follow the distribution: chi-square-free check on the first site's marginal
        P0 = (np.abs(st.amplitudes()) ** 2).reshape(d, -1).sum(axis=1)
        P0 = P0 / P0.sum()
        big = U1MPS.sample_fock(st, rng.random((4000, M)))[0]
        freq = np.bincount(big[:, 0], minlength=d) / 4000.0
        assert np.max(np.abs(freq - P0)) < 5.0 * np.sqrt(0.25 / 4000.0)
    prod = U1MPS.product_state(M, d, N, 4, occ)
    pat, logp, _ = prod.sample_fock(rng.random((5, M)))
    assert np.array_equal(pat, np.tile(occ, (5, 1))) and np.all(np.abs(logp) < 1e-14)
