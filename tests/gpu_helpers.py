"""Helpers for the `-m gpu` parity tests: move states between the oracle and the CUDA library."""
import numpy as np

from u1mps_oracle import U1MPS as Oracle


def make_gpu(M, d, N, chi, **kw):
    from paper_2303_11409_b200.binding import U1MPS
    return U1MPS(M, d, N, chi, **kw)


def gpu_to_oracle(gpu) -> Oracle:
    """Export the whole device state into an oracle object (so that the oracle's validators can be run on it)."""
    st = Oracle(gpu.M, gpu.d, gpu.N, gpu.chi)
    for k in range(gpu.M + 1):
        lam = gpu.export_bond(k)
        st.sectors[k] = sorted(lam)
        st.lam[k] = lam
    for s in range(gpu.M):
        st.gam[s] = gpu.export_site(s)
    st.log_norm = gpu.log_norm()
    return st


def oracle_to_gpu(ora: Oracle, gpu, bonds=None, sites=None):
    bonds = range(ora.M + 1) if bonds is None else bonds
    sites = range(ora.M) if sites is None else sites
    for k in bonds:
        gpu.import_bond(k, ora.lam[k])
    for s in sites:
        gpu.import_site(s, ora.gam[s])


def compare_gate(gpu, ora_pre: Oracle, s, U, chi, cutoff, tol_sigma=1e-10, tol_theta=1e-10, check_theta=True):
    """Teacher-forced parity of ONE gate (SURVEY §8(c) parity protocol (1)).

    gpu must already hold ora_pre's bonds s..s+2 and sites s, s+1.  Applies the gate on both,
    compares a1 (candidates, shapes) bit-exact, a2 Theta(c), a3 sigma and V sigma W, a4 keep(c),
    a5 lambda.  Returns the oracle's GateRecord.  ora_pre is advanced in place.
    """
    rec = ora_pre.apply_gate(s, U, chi=chi, cutoff=cutoff, record=True)
    if check_theta:
        gpu.stage_theta(s, U)
        info = gpu.staged_info()
        assert [c for c, _, _ in info] == rec.charges
        for c, rows, cols in info:
            assert (rows, cols) == rec.theta[c].shape
            th = gpu.export_staged_theta(c, rows, cols)
            scale = max(np.linalg.norm(rec.theta[c]), 1e-300)
            assert np.linalg.norm(th - rec.theta[c]) <= 1e-13 * max(scale, 1e-3), (c, np.linalg.norm(th - rec.theta[c]), scale)
        gpu.stage_svd()
    else:
        gpu.apply_two_site_gate(s, U)
        info = gpu.staged_info()
        assert [c for c, _, _ in info] == rec.charges
    sig1 = max(float(rec.sigma[c][0]) for c in rec.charges)
    fro = np.sqrt(sum(np.linalg.norm(rec.theta[c]) ** 2 for c in rec.charges))
    dev = 0.0   # largest observed |sigma_gpu - sigma_oracle| of this gate
    for c, rows, cols in info:
        V, S, W = gpu.export_staged_svd(c, rows, cols)
        assert np.all(np.diff(S) <= 0), "sigma not descending"
        assert np.max(np.abs(S - rec.sigma[c])) <= tol_sigma * sig1, (c, np.max(np.abs(S - rec.sigma[c])), sig1)
        dev = max(dev, float(np.max(np.abs(S - rec.sigma[c]))))
        recon = (V * S[None, :]) @ W
        assert np.linalg.norm(recon - rec.theta[c]) <= tol_theta * fro, (c, np.linalg.norm(recon - rec.theta[c]), fro)
        # singular vectors above the cutoff - every vector that can be kept - are orthonormal (V, W isometries, pin
        # P4's basis), however small their singular value is
        big = S > cutoff
        if np.any(big):
            Vb, Wb = V[:, big], W[big, :]
            assert np.linalg.norm(Vb.conj().T @ Vb - np.eye(Vb.shape[1])) <= 1e-9
            assert np.linalg.norm(Wb @ Wb.conj().T - np.eye(Wb.shape[0])) <= 1e-9
    gpu.truncate(s, chi, cutoff)
    # a4: kept counts bit-exact unless there is a near-tie at the cut (reading S8: |sigma_chi - sigma_chi+1|
    # <= 1e-10 sigma_1).  At the absolute cutoff (S7) the decision sigma > cutoff can only differ if an oracle
    # sigma lies within the observed GPU/oracle deviation of the cutoff (exact zeros of a rank-deficient
    # Theta come out ~1e-17 on both sides and are not ties) - and only matters where the cutoff, not chi, ends the
    # kept list (fewer than chi values kept, or the chi-th value itself at the cutoff).
    n_kept = sum(rec.keep.values())
    cutoff_binds = n_kept < chi or rec.sigma_chi - cutoff <= 2.0 * dev
    near_tie = ((rec.sigma_next > 0 and abs(rec.sigma_chi - rec.sigma_next) <= 1e-10 * sig1)
                or (rec.cutoff_gap <= 2.0 * dev and cutoff_binds))
    got = dict(gpu.bond_info(s + 1))
    want = {c: k for c, k in rec.keep.items() if k > 0}
    if not near_tie:
        assert got == want, (got, want)
        lam = gpu.export_bond(s + 1)
        for c in want:
            assert np.max(np.abs(lam[c] - ora_pre.lam[s + 1][c])) <= tol_sigma * max(1.0, sig1), c
    else:
        # several kept sets are correct: compare what is unique.  Per sector the counts may differ by at most the
        # number of oracle values that are undecidable (within the observed deviation of the cutoff, or tied with the
        # chi-th value); everything else must agree.
        slack = max(2.0 * dev, 1e-10 * sig1)
        for c in rec.charges:
            sg = rec.sigma[c]
            amb = int(np.sum(np.abs(sg - cutoff) <= 2.0 * dev)) + int(np.sum(np.abs(sg - rec.sigma_chi) <= slack))
            assert abs(got.get(c, 0) - want.get(c, 0)) <= amb, (c, got.get(c, 0), want.get(c, 0), amb)
        assert sum(got.values()) <= chi
    if not near_tie:
        assert_canonical(gpu, s)
    return rec, near_tie


def assert_canonical(gpu, s, tol=1e-9):
    """Pin P4 on what the a5 kernel wrote (the device-side 1/sigma and 1/lambda divisions): per sector c of the rebuilt
    bond s+1, sum_cl (lam Gamma~[s])^H (lam Gamma~[s]) = I and sum_cr (Gamma~[s+1] lam)(Gamma~[s+1] lam)^H = I
    (Eq.12-14: V and W are isometries)."""
    lamL, lamC, lamR = gpu.export_bond(s), gpu.export_bond(s + 1), gpu.export_bond(s + 2)
    gA, gB = gpu.export_site(s), gpu.export_site(s + 1)
    worst = 0.0
    for c, lc in lamC.items():
        k = len(lc)
        accL = np.zeros((k, k), dtype=np.complex128)
        for (cl, cc), blk in gA.items():
            if cc == c:
                a = lamL[cl][:, None] * blk
                accL += a.conj().T @ a
        accR = np.zeros((k, k), dtype=np.complex128)
        for (cc, cr), blk in gB.items():
            if cc == c:
                b = blk * lamR[cr][None, :]
                accR += b @ b.conj().T
        worst = max(worst, np.linalg.norm(accL - np.eye(k)), np.linalg.norm(accR - np.eye(k)))
    assert worst <= tol, worst
    return worst
