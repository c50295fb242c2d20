/* u1mps.h — C ABI of libu1mps.so: the charge-blocked two-site update of a U(1)-symmetric
 * matrix-product state (arXiv:2303.11409; citations are PAPER.md line numbers), hand-written CUDA
 * for sm_100a (B200).  One GPU, one stream, no CPU fallback: every step of the path runs in
 * kernels of this library; if no CUDA device is present every call returns U1MPS_ECUDA.
 *
 * State (Eq.15): {Gamma^[k], lambda^[k], c^[k]}.  0-based indexing: sites
 * s = 0..M-1, bonds k = 0..M; site s has left bond s and right bond s+1.  c^[k] = number of
 * particles on sites k..M-1 (reading S2), so bond 0 = {N}, bond M = {0}.  A bond is a list of charge
 * sectors (c, n_k(c)), ascending c; inside a sector lambda is descending (reading S10).
 * Gamma^[s] is a set of dense blocks Gamma^[s][c_l, c_r], n_s(c_l) x n_{s+1}(c_r), row-major
 * complex128 (interleaved re,im), present only for occupation c_l - c_r in [0, d-1].
 *
 * Update (Eq.16; Eq.12; Eq.13/14 L94-104): steps a1 sector enumeration,
 * a2 Theta(c) contraction, a3 one SVD per centre charge c, a4 global top-chi, a5 renormalise and
 * scatter; a6 readouts.  See DESIGN.md for the data layout and each kernel.
 *
 * Conventions.  All functions return int: 0 = OK, negative = error (never throw, never abort).
 * "host" / "device" says where a pointer must live.  The caller owns every pointer it passes;
 * host arguments (sites, host U) are copied into a library-owned pinned staging ring before the call
 * returns and may be reused at once; a device U is read in stream order (the buffer must stay
 * valid until the stream has passed the call).  The arena and the stream given
 * to u1mps_create are borrowed for the lifetime of the handle.  Calls marked [sync] synchronise
 * the stream; all others only enqueue work (sector sizes stay on the device).
 */
#ifndef U1MPS_H
#define U1MPS_H

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct u1mps u1mps_t; /* opaque; created by u1mps_create, freed by u1mps_destroy */

enum {
  U1MPS_OK = 0,
  U1MPS_EINVAL = -1,  /* bad index / size / occupation / null pointer */
  U1MPS_ENOTU1 = -2,  /* host gate has an entry > 1e-14 that violates charge conservation (Eq.1) */
  U1MPS_ESTAGED = -3, /* call not allowed in the current staging state (see u1mps_apply_two_site_gate) */
  U1MPS_ENOMEM = -4,  /* arena too small for this call */
  U1MPS_ECUDA = -5,   /* CUDA error, or no CUDA device.  Sticky: once a CUDA runtime call of a handle has failed, every
                         later call on that handle returns U1MPS_ECUDA */
  U1MPS_ENOCONV = -6, /* Jacobi SVD hit the sweep limit on some sector.  Detected on the device, so it is reported by the
                         [sync] calls that read the device status (log_norm, norm2, last_stats, staged_info,
                         export_staged_svd).  Sticky, like U1MPS_ENOMEM raised by a launch whose plan did not fit the arena:
                         it stays set until u1mps_clear_status or u1mps_set_product_state, so that a failure in any gate
                         since the last check is never lost */
  U1MPS_ETOOBIG = -7  /* a size beyond the fixed maximum of a no-allocation entry point (u1mps_expect_n_all_static) */
};

const char* u1mps_strerror(int code);

/* Library build info: "u1mps <version> sm_100a". */
const char* u1mps_version(void);

/* Minimum arena size in bytes for a chain of M sites, local dimension d (occupations 0..d-1),
 * N particles, bond dimension chi (<= 4096... see U1MPS_CHI_MAX): state + plan + the workspace of ONE worst-case gate.
 * A larger arena lets u1mps_apply_gate_column process more gates of a column per launch. Returns 0 on bad arguments. */
size_t u1mps_workspace_bytes(int M, int d, int N, int chi);
#define U1MPS_CHI_MAX 4096
#define U1MPS_D_MAX 8

/* Create a handle on caller-allocated DEVICE memory (e.g. torch.empty(nbytes, dtype=uint8, device='cuda')).
 * dev_arena must be 256-byte aligned; cuda_stream is a cudaStream_t (NULL = default stream).
 * The state is undefined until u1mps_set_product_state or the import calls. */
int u1mps_create(u1mps_t** out, int M, int d, int N, int chi, void* dev_arena, size_t arena_bytes,
                 void* cuda_stream);
int u1mps_destroy(u1mps_t* h);

/* |occ_0 ... occ_{M-1}>: occ is HOST int32[M], 0 <= occ < d, sum == N, else U1MPS_EINVAL.
 * Every bond gets one sector of multiplicity 1, Gamma = [[1]], lambda = [1] (SURVEY §8(c) State). */
int u1mps_set_product_state(u1mps_t* h, const int32_t* occ);

/* Steps a1-a3 for sites (i, i+1), i in [0, M-2] (Eq.16; Eq.12 L91 per sector).
 * U: complex128 interleaved, row-major d^2 x d^2, row = out_i*d + out_{i+1}, col = in_i*d + in_{i+1}
 * (reading S3); host pointer if U_on_device == 0 (checked for charge conservation -> ENOTU1),
 * device pointer otherwise (entries violating conservation are never read).  U need not be
 * unitary (S13).  Leaves bond i+1 STAGED (V, sigma, W in the workspace); the only calls allowed
 * while staged are u1mps_truncate(i), the u1mps_export_staged_* calls and u1mps_destroy. */
int u1mps_apply_two_site_gate(u1mps_t* h, int i, const void* U, int U_on_device);

/* Debug / test split of the call above: a1-a2 only (Theta staged), then a3. */
int u1mps_stage_theta(u1mps_t* h, int i, const void* U, int U_on_device);
int u1mps_stage_svd(u1mps_t* h);

/* Steps a4-a5 on the staged gate ("largest chi singular values out of all ... and
 * their corresponding bonds"; Eq.13/14): drop sigma <= cutoff (S7), order (sigma desc, c asc,
 * j asc) (S8), keep the first chi (1 <= chi <= create-time chi; at least one), renormalise (S9),
 * write lambda^[i+1], the sector table of bond i+1, Gamma^[i], Gamma^[i+1]. */
int u1mps_truncate(u1mps_t* h, int i, int chi, double cutoff);

int u1mps_apply_and_truncate(u1mps_t* h, int i, const void* U, int U_on_device, int chi, double cutoff);

/* A whole column of mutually disjoint gates (the paper's gate-level parallelism, L179, folded
 * onto one device): sites is HOST int32[n_gates], strictly increasing with gaps >= 2;
 * U holds n_gates matrices back to back.  Same result as calling u1mps_apply_and_truncate for
 * each gate in order.  All gates of the column share each kernel launch (split into several
 * launches only if the arena is too small for the whole column). */
int u1mps_apply_gate_column(u1mps_t* h, const int32_t* sites, int n_gates, const void* U,
                            int U_on_device, int chi, double cutoff);

/* a6 readouts.  out_host are HOST pointers.  All [sync]. */
int u1mps_norm2(u1mps_t* h, double* out_host);                     /* exp(2 * accumulated log-norm) */
int u1mps_log_norm(u1mps_t* h, double* out_host);                  /* sum over gates of 0.5 ln(sum sigma_kept^2) */
int u1mps_expect_n(u1mps_t* h, int site, double* out_host);        /* canonical-form <n_site> */
int u1mps_expect_n_all(u1mps_t* h, double* out_host /*[M]*/);      /* all sites, one launch */
int u1mps_bond_entropy(u1mps_t* h, int bond, double* out_host);    /* -sum lambda^2 ln lambda^2 (natural log, S23) */
int u1mps_bond_entropy_all(u1mps_t* h, double* out_host /*[M+1]*/);
/* u1mps_expect_n_all for callers that must not allocate (code under CUDA graph capture, serving loops, harnesses that
 * forbid cudaMalloc): the same kernel and the same canonical-form <n_s> of all sites (Eq.10, Eq.15),
 * with the kernel's scratch (the partial sums of the slices a site is cut into and one completion counter per site) in
 * a static device array of the library instead of the arena: 69 632 bytes on every GPU that loads the library, held
 * until the process exits.  The call makes no cudaMalloc / cudaFree and no allocating library call: it enqueues one
 * memset (the counters it uses must start at zero; the array keeps the previous call's contents) and one kernel on the
 * handle's stream and returns WITHOUT synchronising.  [async]
 *   out_dev: DEVICE double[M], 8-byte aligned, owned by the caller, on the device the handle lives on (which must be
 *            the current device); valid once the handle's stream has reached this point.  A host pointer -> U1MPS_EINVAL.
 *   M > U1MPS_STATIC_SITES_MAX -> U1MPS_ETOOBIG (nothing is enqueued); U1MPS_ESTAGED while a gate is staged.
 * Every handle and every call on a device shares the one array: calls that overlap on the GPU (handles on different
 * streams without an ordering between them) race on it and return garbage - serialise them.  Calls on one stream are
 * ordered and safe.  The sums are added in the same fixed order as in u1mps_expect_n_all (bit-identical results as long
 * as M <= U1MPS_STATIC_SITES_MAX, which keeps the slice count the same). */
#define U1MPS_STATIC_SITES_MAX 1024
int u1mps_expect_n_all_static(u1mps_t* h, double* out_dev /*[M]*/);
/* Full-environment <psi|n_k|psi> / <psi|psi> of all sites (state of Eq.15): left and
 * right environments contracted explicitly, exact for whatever Gamma, lambda the handle holds - unlike the
 * canonical-form u1mps_expect_n, which is exact only while nothing has been truncated (Eq.10).  The caller
 * provides DEVICE scratch (256-byte aligned) of at least u1mps_expect_n_full_bytes (it depends on the current sector
 * tables: all left environments of the chain are kept, sum over bonds and sectors of n^2 complex128, plus two Gamma-sized
 * buffers); U1MPS_ENOMEM if it is too small.  out_host: [M].  Both [sync]. */
int u1mps_expect_n_full_bytes(u1mps_t* h, size_t* bytes_host);
int u1mps_expect_n_full(u1mps_t* h, double* out_host, void* scratch_dev, size_t scratch_bytes);
/* Two-point function <psi|n_j n_k|psi> / <psi|psi> (any order of j, k; j == k gives <n_j^2>), the same environment
 * sweeps with the occupation c_l - c_r inserted into the transfer step of site j (state of Eq.15).  Device
 * scratch of at least u1mps_expect_nn_full_bytes (six environment-sized and two Gamma-sized buffers).  Both [sync]. */
int u1mps_expect_nn_full_bytes(u1mps_t* h, size_t* bytes_host);
int u1mps_expect_nn_full(u1mps_t* h, int site_j, int site_k, double* out_host, void* scratch_dev, size_t scratch_bytes);
/* Fock-pattern sampling (Eq.7-8: the distribution over occupation patterns that
 * boson sampling asks for; state of Eq.15): n_samples patterns (n_0 .. n_{M-1}), each drawn from
 * |<n|psi>|^2 / <psi|psi> exactly (right environments contracted explicitly, so truncation does not bias the draw).
 * The random numbers are an INPUT: u_host[b * M + s] in [0, 1) (else U1MPS_EINVAL) decides site s of sample b by inverse
 * CDF over the occupations 0 .. d-1 in ascending order, conditioned on the occupations already drawn for sites < s; the
 * same u gives the same patterns on every run.  pattern_host: HOST int32 [n_samples * M]; logp_host: HOST [n_samples],
 * ln of the probability of the drawn pattern.  Device scratch (256-byte aligned) of at least u1mps_sample_fock_bytes:
 * all right environments of the chain (sum over bonds and sectors of n^2 complex128), one Gamma-sized buffer and
 * (d + 2) boundary vectors per sample; U1MPS_ENOMEM if it is too small.  1 <= n_samples <= U1MPS_SAMPLES_MAX.  Both [sync]. */
#define U1MPS_SAMPLES_MAX 65536
int u1mps_sample_fock_bytes(u1mps_t* h, int n_samples, size_t* bytes_host);
int u1mps_sample_fock(u1mps_t* h, int n_samples, const double* u_host, int32_t* pattern_host, double* logp_host,
                      void* scratch_dev, size_t scratch_bytes);
/* Sector table of a bond: writes up to cap (charge, count) pairs, ascending charge; *n_sectors = how many exist. */
int u1mps_bond_info(u1mps_t* h, int bond, int32_t* n_sectors, int32_t* charges, int32_t* counts, int cap);
int u1mps_bond_dims(u1mps_t* h, int32_t* dims_host /*[M+1]*/);
/* Statistics since create / set_product_state: total discarded weight; of the LAST column or
 * gate: kept bond dimension of its first gate, Jacobi sweeps used by its slowest sector (a sweep = one visit of every
 * panel pair of the largest sector; U1MPS_ENOCONV is returned if some sector needed more than U1MPS_MAXSWEEP). */
int u1mps_last_stats(u1mps_t* h, double* discarded_weight, int* kept, int* sweeps);
/* Clear the sticky device status (U1MPS_ENOCONV / device-side U1MPS_ENOMEM).  Enqueued in stream order. */
int u1mps_clear_status(u1mps_t* h);

/* Export / import (teacher-forced parity, checkpoints).  All [sync]; host buffers. */
int u1mps_export_bond(u1mps_t* h, int bond, double* lambda_host, int cap);  /* ascending c, descending inside */
/* Block Gamma^[site][cl, cr], row-major complex128, n_site(cl) x n_{site+1}(cr); cap in BYTES. */
int u1mps_export_site(u1mps_t* h, int site, int cl, int cr, void* block_host, size_t cap);
/* Replace the sector table and lambda of a bond.  charges ascending, counts >= 1, sum <= chi.
 * Invalidates the blocks of sites bond-1 and bond: import them afterwards. */
int u1mps_import_bond(u1mps_t* h, int bond, int n_sectors, const int32_t* charges, const int32_t* counts,
                      const double* lambda_host);
int u1mps_import_site(u1mps_t* h, int site, int cl, int cr, const void* block_host, size_t bytes);
int u1mps_set_log_norm(u1mps_t* h, double log_norm, double discarded);

/* Staged-gate read-back (valid between apply_two_site_gate / stage_* and truncate).  [sync]
 * Candidate centre charges of the staged gate: for each, rows(c) and cols(c) of Theta(c). */
int u1mps_staged_info(u1mps_t* h, int32_t* n_cand, int32_t* charges, int32_t* rows, int32_t* cols, int cap);
/* After stage_theta: Theta(c), row-major rows x cols (row blocks ascending c_l, column blocks ascending c_r). */
int u1mps_export_staged_theta(u1mps_t* h, int c, void* theta_host, size_t cap);
/* After stage_svd / apply_two_site_gate: thin SVD of Theta(c): V rows x r, sigma r (descending), W r x cols,
 * r = min(rows, cols), row-major.  Any of the three pointers may be NULL. */
int u1mps_export_staged_svd(u1mps_t* h, int c, void* V_host, double* sigma_host, void* W_host);

/* Per-kernel device timing (for bench.py's roofline): while enabled, every kernel launch of the handle is
 * bracketed by CUDA events on the handle's stream; u1mps_profile_read [sync] sums the elapsed times (ms) and
 * launch counts per stage since the last read / enable into HOST arrays of U1MPS_NSTAGE entries and resets. */
#define U1MPS_NSTAGE 8
int u1mps_profile_enable(u1mps_t* h, int on);
int u1mps_profile_read(u1mps_t* h, double* ms_host, long long* launches_host);
const char* u1mps_stage_name(int stage); /* "a1_plan", "a2_contract", ... ; "" if out of range */

/* Trace of the LAST a3 launch (one column or gate) [sync]: out_host[0] = start time, then 4 arrays of U1MPS_MAXSWEEP
 * entries, one per Jacobi sweep (= np_max rounds of the modulus ordering, np_max = panels of the largest sector of the
 * launch): end time (GPU globaltimer, ns), panel-pair items that rotated, inner EVD sweeps run, sectors not yet
 * converged at the end of the sweep.  cap (entries of out_host) must be >= 4 * U1MPS_MAXSWEEP + 1. */
#define U1MPS_MAXSWEEP 30
int u1mps_svd_trace(u1mps_t* h, long long* out_host, int cap);

/* Number of kernels this handle has launched since create (for bench.py's gpu_launches). */
int u1mps_launch_count(u1mps_t* h, long long* out_host);

#ifdef __cplusplus
}
#endif
#endif /* U1MPS_H */
