"""Seeded synthetic inputs: gate generators and the five workload recipes of BASELINE.json.

This module is the ONLY code shared by the CPU oracle (tests) and the CUDA path (bench, tests).
It builds input arrays (two-site gate matrices, occupation strings, gate schedules) and holds
none of the method's arithmetic (no contraction, SVD, truncation or readout).

Conventions (reading S3 of DESIGN.md): a two-site gate is a complex128
matrix U[(out_a*d + out_b), (in_a*d + in_b)] of shape (d*d, d*d) acting on sites (s, s+1);
a U(1) gate has U[r, c] == 0 unless out_a + out_b == in_a + in_b (Eq.1).

Recipes follow SURVEY.md §8(d) "Inputs": seed = 230311409 + config index (1-based),
numpy.random.default_rng, gates drawn column by column, left to right.
"""
from __future__ import annotations

import math
from dataclasses import dataclass
from typing import Iterator, List, Tuple

import numpy as np

SEED_BASE = 230311409


# --------------------------------------------------------------------------------------
# gate generators
# --------------------------------------------------------------------------------------
def haar_2x2(rng: np.random.Generator) -> np.ndarray:
    """2x2 Haar unitary: complex Ginibre -> QR -> fix column phases by the phase of diag(R)."""
    z = (rng.standard_normal((2, 2)) + 1j * rng.standard_normal((2, 2))) / math.sqrt(2.0)
    q, r = np.linalg.qr(z)
    ph = np.diag(r) / np.abs(np.diag(r))
    return q * ph[None, :]


def hardcore_haar_gate(rng: np.random.Generator) -> np.ndarray:
    """d=2 gate 1 (+) Haar(2x2) (+) 1 in the n_a+n_b basis (configs 1-2 of BASELINE.json).

    Basis index = n_a*2 + n_b: |00>, |01>, |10>, |11>; the Haar block mixes |01>, |10>.
    """
    u = np.zeros((4, 4), dtype=np.complex128)
    u[0, 0] = 1.0
    u[3, 3] = 1.0
    u[1:3, 1:3] = haar_2x2(rng)
    return u


def xxz_gate(delta: float, dt: float) -> np.ndarray:
    """exp(-i dt (sx sx + sy sy + delta sz sz)) with n = (1 - sz)/2 (Eq.3-4).

    Closed form: e^{-i dt delta} on |00>,|11>; e^{+i dt delta} [[cos 2dt, -i sin 2dt],
    [-i sin 2dt, cos 2dt]] on span{|01>,|10>}.  tests/ checks it against scipy expm of the 4x4.
    """
    u = np.zeros((4, 4), dtype=np.complex128)
    u[0, 0] = u[3, 3] = np.exp(-1j * dt * delta)
    ph = np.exp(1j * dt * delta)
    c, s = math.cos(2.0 * dt), math.sin(2.0 * dt)
    u[1, 1] = u[2, 2] = ph * c
    u[1, 2] = u[2, 1] = ph * (-1j * s)
    return u


def beam_splitter_2x2(theta: float, phi: float) -> np.ndarray:
    """Mode unitary u = [[cos t, -e^{-i phi} sin t], [e^{i phi} sin t, cos t]]; a_j^+ -> sum_k u[k,j] a_k^+."""
    c, s = math.cos(theta), math.sin(theta)
    return np.array([[c, -np.exp(-1j * phi) * s], [np.exp(1j * phi) * s, c]], dtype=np.complex128)


def beam_splitter_gate(u: np.ndarray, d: int) -> np.ndarray:
    """Fock-space matrix of a two-mode linear-optical unitary, occupations restricted to 0..d-1.

    <m1,m2|B|n1,n2> = sqrt(m1! m2! / (n1! n2!)) * sum_{p+q=m1} C(n1,p) C(n2,q)
                      u11^p u21^(n1-p) u12^q u22^(n2-q)            (Eq.8)
    Block-diagonal in n1+n2.  Entries with any occupation > d-1 are dropped (reading S6), so
    the restricted gate is unitary only on total photon number <= d-1.
    """
    g = np.zeros((d * d, d * d), dtype=np.complex128)
    u11, u12, u21, u22 = u[0, 0], u[0, 1], u[1, 0], u[1, 1]
    for n1 in range(d):
        for n2 in range(d):
            n = n1 + n2
            for m1 in range(max(0, n - (d - 1)), min(d - 1, n) + 1):
                m2 = n - m1
                acc = 0.0 + 0.0j
                for p in range(max(0, m1 - n2), min(n1, m1) + 1):
                    q = m1 - p
                    acc += (math.comb(n1, p) * math.comb(n2, q)
                            * u11 ** p * u21 ** (n1 - p) * u12 ** q * u22 ** (n2 - q))
                pref = math.sqrt(math.factorial(m1) * math.factorial(m2)
                                 / (math.factorial(n1) * math.factorial(n2)))
                g[m1 * d + m2, n1 * d + n2] = pref * acc
    return g


def haar_beam_splitter_gate(rng: np.random.Generator, d: int) -> np.ndarray:
    """phi ~ U[0,2pi), cos^2(theta) ~ U[0,1] (2x2 Haar measure on the transmission; reading R-BS)."""
    phi = rng.uniform(0.0, 2.0 * math.pi)
    theta = math.acos(math.sqrt(rng.uniform(0.0, 1.0)))
    return beam_splitter_gate(beam_splitter_2x2(theta, phi), d)


def swap_gate(d: int) -> np.ndarray:
    g = np.zeros((d * d, d * d), dtype=np.complex128)
    for a in range(d):
        for b in range(d):
            g[b * d + a, a * d + b] = 1.0
    return g


def random_u1_gate(rng: np.random.Generator, d: int, unitary: bool = True) -> np.ndarray:
    """Generic charge-conserving gate: an independent random (Haar or Ginibre) block per n_a+n_b."""
    g = np.zeros((d * d, d * d), dtype=np.complex128)
    for n in range(2 * d - 1):
        idx = [a * d + (n - a) for a in range(d) if 0 <= n - a < d]
        k = len(idx)
        z = (rng.standard_normal((k, k)) + 1j * rng.standard_normal((k, k))) / math.sqrt(2.0)
        if unitary:
            q, r = np.linalg.qr(z)
            z = q * (np.diag(r) / np.abs(np.diag(r)))[None, :]
        g[np.ix_(idx, idx)] = z
    return g


# --------------------------------------------------------------------------------------
# workload recipes (BASELINE.json configs 1-5)
# --------------------------------------------------------------------------------------
@dataclass(frozen=True)
class Workload:
    index: int            # 1-based config index of BASELINE.json
    name: str
    M: int
    d: int
    N: int
    chi: int
    cutoff: float
    occ: Tuple[int, ...]  # initial product state, site 0 first
    family: str           # "haar2" | "xxz" | "bs"
    columns: int          # number of gate columns (a brick-wall layer = 2 columns)
    delta: float = 0.5
    dt: float = 0.05

    @property
    def seed(self) -> int:
        return SEED_BASE + self.index

    @property
    def n_gates(self) -> int:
        return sum(len(column_sites(self.M, t)) for t in range(self.columns))


def _alternating(M: int, first: int) -> Tuple[int, ...]:
    return tuple((first + s) % 2 for s in range(M))


WORKLOADS = {
    1: Workload(1, "hcb-M16-chi32", 16, 2, 8, 32, 1e-12, _alternating(16, 1), "haar2", 2),
    2: Workload(2, "hcb-M64-chi256", 64, 2, 32, 256, 1e-12, _alternating(64, 1), "haar2", 40),
    3: Workload(3, "xxz-M128-chi1024", 128, 2, 64, 1024, 1e-12, _alternating(128, 0), "xxz", 100),
    4: Workload(4, "bs-M32-d5-chi512", 32, 5, 16, 512, 1e-12,
                tuple([1] * 16 + [0] * 16), "bs", 32),
    5: Workload(5, "bs-M100-d4-chi4096", 100, 4, 50, 4096, 1e-12, _alternating(100, 1), "bs", 100),
}


def column_sites(M: int, t: int) -> List[int]:
    """Left sites s of the disjoint gates (s, s+1) in column t: s = t%2, t%2+2, ... <= M-2 (reading S15)."""
    return list(range(t % 2, M - 1, 2))


def gate_columns(w: Workload, max_columns: int | None = None) -> Iterator[Tuple[np.ndarray, np.ndarray]]:
    """Yield (sites[int32, g], U[complex128, g, d*d, d*d]) for each column of the workload, in order."""
    rng = np.random.default_rng(w.seed)
    ncol = w.columns if max_columns is None else min(w.columns, max_columns)
    xxz = xxz_gate(w.delta, w.dt) if w.family == "xxz" else None
    for t in range(ncol):
        sites = column_sites(w.M, t)
        us = np.empty((len(sites), w.d * w.d, w.d * w.d), dtype=np.complex128)
        for g in range(len(sites)):
            if w.family == "haar2":
                us[g] = hardcore_haar_gate(rng)
            elif w.family == "xxz":
                us[g] = xxz
            elif w.family == "bs":
                us[g] = haar_beam_splitter_gate(rng, w.d)
            else:  # pragma: no cover
                raise ValueError(w.family)
        yield np.asarray(sites, dtype=np.int32), us


def small_variant(w: Workload, M: int, N: int, chi: int, columns: int, occ=None) -> Workload:
    """Same gate family and seed, smaller chain: used by tests so that the oracle finishes in seconds."""
    if occ is None:
        if w.family == "bs" and w.index == 4:
            occ = tuple([1] * N + [0] * (M - N))
        else:
            occ = tuple(w.occ[:M])
    assert sum(occ) == N and len(occ) == M
    return Workload(w.index, w.name + f"-small-M{M}", M, w.d, N, chi, w.cutoff, tuple(occ), w.family,
                    columns, w.delta, w.dt)


# --------------------------------------------------------------------------------------
# synthetic saturated-bond state for per-gate parity tests and the per-gate microbenchmark
# (parabolic sector profile, random blocks, geometric lambda inside a sector)
# --------------------------------------------------------------------------------------
def parabolic_profile(chi: int, R: int) -> List[int]:
    """R sector sizes ~ 1 - ((x - x0)/((R+1)/2))^2, each >= 1, summing exactly to chi."""
    x0 = (R - 1) / 2.0
    w = np.array([1.0 - ((x - x0) / ((R + 1) / 2.0)) ** 2 for x in range(R)])
    n = np.maximum(1, np.floor(w / w.sum() * chi).astype(int))
    i = 0
    while n.sum() < chi:
        n[(R // 2 + i) % R] += 1
        i += 1
    while n.sum() > chi:
        j = int(np.argmax(n))
        n[j] -= 1
    return [int(v) for v in n]


# sector sizes of a saturated bond of config 3 (XXZ, chi = 1024) as measured on the trajectory after 50 layers
# (DESIGN.md section 4); used so that the CPU-baseline sample has the block sizes of the real workload
SATURATED_PROFILE = {3: (5, 32, 100, 195, 256, 229, 139, 54, 13, 1),
                     # config 5 (beam splitters, d = 4, chi = 4096), bond 50 after 16 columns
                     5: (2, 18, 77, 229, 460, 686, 809, 758, 550, 311, 138, 47, 10, 1)}


def synthetic_gate_state(d: int, chi: int, R: int, seed: int, decay: float = 0.97, profile=None):
    """Random three-bond neighbourhood for one gate on sites (2, 3) of a short chain (M >= 6).

    Returns (M, N, site, lam, gam): lam[k] = {c: descending positive vector} for bonds 2, 3, 4;
    gam[s] = {(cl, cr): random complex block} for sites 2, 3.  Bond k's sector charges are
    c0_k .. c0_k + R - 1 with c0 dropping by (d - 1) // 2 + (d % 2 == 0) per bond, so that every
    occupation 0..d-1 occurs.  No arithmetic of the method is done here: the blocks are plain
    random numbers (the update is defined for any Gamma and any positive lambda).
    """
    rng = np.random.default_rng(seed)
    site = 2
    step = max(1, d // 2)
    if profile is not None:
        R = len(profile)
    N0 = R + 4 * step + 2
    first = {k: max(0, N0 - 2 - (k - 1) * step - R // 2 + 1) for k in (2, 3, 4)}
    N = max(N0, first[2] + R - 1)          # every sector charge must lie in [0, N]
    M = max(6, -(-N // (d - 1)) + 1)
    prof = list(profile) if profile is not None else parabolic_profile(chi, R)
    lam, gam = {}, {}
    for k in (2, 3, 4):
        c0 = first[k]
        lk = {}
        for x, n in enumerate(prof):
            v = np.sort(rng.uniform(0.5, 1.0, n) * decay ** np.arange(n))[::-1]
            lk[c0 + x] = v
        tot = math.sqrt(sum(float(np.sum(v ** 2)) for v in lk.values()))
        lam[k] = {c: v / tot for c, v in lk.items()}
    for s in (2, 3):
        gs = {}
        for cl, vl in lam[s].items():
            for cr, vr in lam[s + 1].items():
                if 0 <= cl - cr <= d - 1:
                    nl, nr = len(vl), len(vr)
                    gs[(cl, cr)] = (rng.standard_normal((nl, nr)) + 1j * rng.standard_normal((nl, nr))) / math.sqrt(nl + nr)
        gam[s] = gs
    return M, N, site, lam, gam
