"""Independent pins for the oracle: exact d^M state-vector evolution and textbook closed forms.

Nothing here imports oracle/ or the CUDA path.  Site 0 is the most significant base-d digit.
"""
import itertools
import math

import numpy as np


def product_vector(occ, d):
    idx = 0
    for o in occ:
        idx = idx * d + int(o)
    v = np.zeros(d ** len(occ), dtype=np.complex128)
    v[idx] = 1.0
    return v


def apply_two_site(vec, M, d, s, U):
    """psi'[.., a', b', ..] = sum_{a,b} U[(a' d + b'), (a d + b)] psi[.., a, b, ..] (Eq.11 without the MPS)."""
    t = vec.reshape(d ** s, d * d, d ** (M - s - 2))
    return np.einsum("xy,lyr->lxr", np.asarray(U).reshape(d * d, d * d), t).reshape(-1)


def number_expectation(vec, M, d, s):
    p = np.abs(vec.reshape(d ** s, d, d ** (M - s - 1))) ** 2
    return float(np.einsum("lir,i->", p, np.arange(d))) / float(np.sum(np.abs(vec) ** 2))


def total_charge_weights(vec, M, d):
    """Probability weight per total particle number."""
    out = {}
    for idx in np.nonzero(np.abs(vec) > 0)[0]:
        n, x = 0, int(idx)
        for _ in range(M):
            n += x % d
            x //= d
        out[n] = out.get(n, 0.0) + abs(vec[idx]) ** 2
    return out


def schmidt_values(vec, M, d, k):
    """Singular values across the cut between sites k-1 and k."""
    return np.linalg.svd(vec.reshape(d ** k, d ** (M - k)), compute_uv=False)


def permanent(a):
    n = a.shape[0]
    if n == 0:
        return 1.0 + 0j
    tot = 0j
    for perm in itertools.permutations(range(n)):
        p = 1.0 + 0j
        for i in range(n):
            p *= a[i, perm[i]]
        tot += p
    return tot


def fock_amplitude(Umode, n_in, m_out):
    """<m_out| B |n_in> = perm(U[rows(m), cols(n)]) / sqrt(prod m! prod n!)  with a_j^+ -> sum_k U[k,j] a_k^+ (Eq.8)."""
    rows = [k for k, m in enumerate(m_out) for _ in range(m)]
    cols = [j for j, n in enumerate(n_in) for _ in range(n)]
    if len(rows) != len(cols):
        return 0j
    sub = Umode[np.ix_(rows, cols)]
    norm = math.sqrt(np.prod([math.factorial(m) for m in m_out]) * np.prod([math.factorial(n) for n in n_in]))
    return permanent(sub) / norm
