// svd.cu — step a3: one SVD per centre-charge sector ("Singular value decompositions are
// then performed on each Theta(c^[k])"; Eq.12), for all sectors of all gates of the chunk at once.
// The paper calls a library SVD (L131); here it is a batched one-sided (Hestenes) BLOCK Jacobi SVD:
// the columns of the stacked matrix [G; J] (G = Theta(c) or its conjugate transpose so that
// m >= n, J = identity) are made mutually orthogonal; then sigma_j = |G_j|, left vectors
// G_j / sigma_j, right vectors J_j.
//
// Blocking.  Columns are taken in the order of their initial norms (a norm + sort pre-pass fills the logical ->
// physical column map; the matrix is not permuted) and grouped in panels of U1_PB = 16.  A work item is a panel
// pair P = [Pa Pb] (32 columns):
//   1. Gram   H = P^H P over the m rows of G           (FP64 DMMA.8x8x4 tiles, chunks of 32 rows staged
//                                                        in shared memory by a 2-stage cp.async ring)
//   2. EVD    H = Q diag Q^H by two-sided Jacobi in shared memory (16 disjoint rotations per round on
//             two-by-two units, in place; rotations sort the pair by norm, de Rijk style)
//   3. update [Pa Pb] <- [Pa Pb] Q over all m + n rows  (DMMA again, Q held in registers as B fragments)
// A persistent cooperative grid walks the panel pairs of every sector in lock step, one grid sync per round, items
// handed out through an atomic ticket.  Round t pairs the panels with (i + j) mod np == (t + 1) mod np (modulus
// ordering: a software-pipelined cyclic-by-rows ordering; with the norm-sorting rotations it deflates a graded
// spectrum from the top like a Gram-Schmidt pass, and needs about 2/3 of the sweeps of the round-robin tournament
// on the Theta blocks of the workloads).  Convergence is decided on the device per sector (np consecutive rounds,
// i.e. every panel pair once, without an off-diagonal Gram entry above the threshold), no host round trip.
#ifdef SV_PROFILE
#include <cstdlib>
#endif
#include "common.cuh"

#define SV_W 32                      // columns of a pair item
#define SV_R 32                      // rows per staged chunk
#define SV_LDG 36                    // shared-memory leading dimension (complex elements) in the Gram phase: 4 mod 8
#define SV_LDU 34                    // ... in the update phase: 2 mod 8 (both: conflict-free LDS.128 fragment loads)
#define SV_STAGE (SV_W * SV_LDG)     // complex elements per stage
#ifndef SV_MIN_ACTIVE
#define SV_MIN_ACTIVE 2                  // a3 throttle: CTAs per SM that take items however little work there is
#endif
#ifndef SV_ITEMS_PER_CTA
#define SV_ITEMS_PER_CTA 4           // a3 throttle: items per active CTA and round below which fewer CTAs per SM are used
#endif
#ifndef SV_NSTAGE
#define SV_NSTAGE 3                  // cp.async ring depth: chunks c + 1 and c + 2 are in flight while chunk c is consumed
#endif
#define SV_HLD 33                    // leading dimension of the 32 x 32 Gram matrix (row-major)
static_assert(U1_MAXSWEEP == 30, "keep U1MPS_MAXSWEEP of include/u1mps.h in step");
#define SV_QLD 36                    // leading dimension of the transposed eigenvector matrix Qt (4 mod 8: B fragments)
#ifndef SV_TOLFAC
#define SV_TOLFAC 8.0                // stopping threshold tol = SV_TOLFAC eps sqrt(m) on |h_pq| / sqrt(h_pp h_qq)
#endif
#ifndef SV_INNER_MAX
#define SV_INNER_MAX 2               // inner EVD sweeps per item (the outer iteration finishes the job; measured best of 1..4)
#endif
#define SV_LASTPASS 1e-18            // (relative off-diagonal)^2 below which a rotation needs no verification sweep
#ifndef SV_QUAD
#define SV_QUAD 1e-4                 // no second inner sweep after one whose largest relative off-diagonal^2 was below this (measured best of 1e-14 .. 3e-1)
#endif
#define SV_GROUP 128                 // threads per pair item (= one CTA: SV_NGROUP == 1; several groups per CTA were tried and dropped)
#define SV_NGROUP (U1_SVD_THREADS / SV_GROUP)
#ifndef SV_CTAS
#define SV_CTAS 4                    // resident CTAs per SM the kernel is compiled for (registers <= 128: no spills with the
                                     // 3M accumulators; measured best of 3..6, profiles/r2_svd_tuning.md)
#endif
#define SV_RING_BYTES (SV_NSTAGE * SV_STAGE * 16)
#define SV_EVD_BYTES ((SV_W * SV_HLD + SV_W * SV_QLD) * 16 + 2 * U1_PB * 32 + SV_W * U1_PB * 2)   // H, Qt, rotations, pivot table
#define SV_SMEM_BYTES (SV_RING_BYTES > SV_EVD_BYTES ? SV_RING_BYTES : SV_EVD_BYTES)   // the EVD buffers alias the idle ring

__device__ __forceinline__ double warp_sum(double v) {
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
  return v;
}

__device__ __forceinline__ void cp_async16(void* smem, const void* gmem, int src_bytes) {
  const unsigned s = (unsigned)__cvta_generic_to_shared(smem);
  asm volatile("cp.async.cg.shared.global [%0], [%1], 16, %2;\n" ::"r"(s), "l"(gmem), "r"(src_bytes) : "memory");
}
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;\n" ::: "memory"); }
template <int N>
__device__ __forceinline__ void cp_async_wait() { asm volatile("cp.async.wait_group %0;\n" ::"n"(N) : "memory"); }

// Trial build -DSV_TMA (profiles/r2_tma_trial.md): the chunk loader as 1-D bulk copies (cp.async.bulk, the TMA engine,
// completion on an mbarrier per ring stage) issued by one warp, instead of 16-byte cp.async by all threads.
struct RingState {
#ifdef SV_TMA
  unsigned long long* bar;   // [SV_NSTAGE] mbarriers in shared memory
  unsigned phase;            // bit s: parity the next wait on stage s expects
#endif
};
#ifdef SV_TMA
__device__ __forceinline__ unsigned smem_u32(const void* p) { return (unsigned)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void mbar_init(unsigned long long* b, int count) {
  asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;\n" ::"r"(smem_u32(b)), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_expect_tx(unsigned long long* b, unsigned bytes) {
  asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;\n" ::"r"(smem_u32(b)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void bulk_g2s(void* dst, const void* src, unsigned bytes, unsigned long long* b) {
  asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];\n"
               ::"r"(smem_u32(dst)), "l"(src), "r"(bytes), "r"(smem_u32(b)) : "memory");
}
__device__ __forceinline__ void mbar_wait(unsigned long long* b, unsigned parity) {
  unsigned ok = 0;
  for (unsigned spins = 0; !ok && spins < (1u << 22); ++spins)   // bounded: a lost completion must not hang the GPU
    asm volatile("{\n .reg .pred p;\n mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n selp.u32 %0, 1, 0, p;\n}\n"
                 : "=r"(ok) : "r"(smem_u32(b)), "r"(parity) : "memory");
}
#endif

// Named barrier of a 128-thread group (id g + 1; 0 is __syncthreads) and its group-wide OR.
__device__ __forceinline__ void gsync(int g) { asm volatile("bar.sync %0, 128;\n" ::"r"(g + 1) : "memory"); }
__device__ __forceinline__ int gsync_or(int g, int pred) {
  int r;
  asm volatile("{\n .reg .pred p, q;\n setp.ne.s32 p, %2, 0;\n bar.red.or.pred q, %1, 128, p;\n selp.s32 %0, 1, 0, q;\n}\n"
               : "=r"(r) : "r"(g + 1), "r"(pred) : "memory");
  return r;
}

struct Item {
  cplx* W;        // stacked (m + n) x n column-major Jacobi matrix of the sector
  int m, mt;      // rows of G; m + n = leading dimension
  int ca, na;     // first column / number of columns of panel a
  int cb, nb;     // ... of panel b (nb = 0: single-panel item)
  const int* col; // [32] shared memory: physical column of each of the item's columns (logical order = sorted by initial norm)
  double tol2;
};

// Stage rows [row0, row0 + SV_R) x the 32 columns of the item into shared memory (column-major, leading dimension ld);
// rows >= rowlim and absent columns are zero-filled.  Thread (r = gtid % 32, it) copies row row0 + r of the columns
// j = gtid / 32 + 4 it; their addresses are worked out once per item (Loader), a chunk only adds its row offset.
struct Loader {
  const cplx* src[SV_W * SV_R / SV_GROUP];   // row r of column j (item's W if the column is absent: never read, 0 bytes copied)
  unsigned ok;                                // bit it: column present
};
__device__ __forceinline__ Loader make_loader(const Item& I, int gtid) {
  Loader L;
  L.ok = 0;
  const int r = gtid & (SV_R - 1);
#pragma unroll
  for (int it = 0; it < SV_W * SV_R / SV_GROUP; ++it) {
    const int j = gtid / SV_R + it * (SV_GROUP / SV_R);
    const bool ok = j < U1_PB ? j < I.na : j - U1_PB < I.nb;
    L.src[it] = ok ? I.W + (long long)I.col[j] * I.mt + r : I.W;
    L.ok |= ok ? (1u << it) : 0u;
  }
  return L;
}
#ifdef SV_TMA
// stage `sidx`: one bulk copy per present column (32 rows x 16 B = 512 B contiguous in global and in shared memory),
// lane j of warp 0 takes column j; ragged tails and absent columns are zero-filled with ordinary stores
__device__ __forceinline__ void load_chunk_tma(cplx* st, int ld, const Item& I, int row0, int rowlim, int gtid, RingState& RS, int sidx) {
  const int rows = min(SV_R, rowlim - row0);
  const int lane = gtid & 31;
  if (gtid < 32) {
    const bool present = lane < U1_PB ? lane < I.na : lane - U1_PB < I.nb;
    const unsigned bytes = present ? (unsigned)rows * 16u : 0u;
    unsigned total = bytes;
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) total += __shfl_xor_sync(0xffffffffu, total, o);
    if (lane == 0) mbar_expect_tx(RS.bar + sidx, total);
    __syncwarp();
    if (present) bulk_g2s(st + lane * ld, I.W + (long long)I.col[lane] * I.mt + row0, bytes, RS.bar + sidx);
  }
  if (rows < SV_R || I.na < U1_PB || I.nb < U1_PB) {
    for (int idx = gtid; idx < SV_W * SV_R; idx += SV_GROUP) {
      const int j = idx / SV_R, r = idx - j * SV_R;
      const bool present = j < U1_PB ? j < I.na : j - U1_PB < I.nb;
      if (!present || r >= rows) st[j * ld + r] = make_double2(0.0, 0.0);
    }
  }
}
#endif
__device__ __forceinline__ void load_chunk(cplx* st, int ld, const Loader& L, int row0, int rowlim, int gtid) {
  const int r = gtid & (SV_R - 1);
  const bool rok = row0 + r < rowlim;
  cplx* dst = st + (gtid / SV_R) * ld + r;
#pragma unroll
  for (int it = 0; it < SV_W * SV_R / SV_GROUP; ++it) {
    const bool ok = rok && ((L.ok >> it) & 1u);
    cp_async16(dst + it * (SV_GROUP / SV_R) * ld, ok ? L.src[it] + row0 : L.src[it], ok ? 16 : 0);
  }
}

// ---- phase 1: H = P^H P over rows [0, m).  H is Hermitian: only the 10 tiles (8 x 8 each) of the upper triangle of
// the 4 x 4 tile grid are computed, 3 + 3 + 2 + 2 per warp: warp 0 (0,0) (0,1) (0,2); warp 1 (3,0) (3,1) (3,2), stored
// as the conjugate transposes (0,3) (1,3) (2,3); warp 2 (1,1) (1,2); warp 3 (2,2) (3,3).
__device__ __forceinline__ void gram_phase(cplx* stages, cplx* Hs, const Item& I, const Loader& L, RingState& RS, int g, int gtid) {
  const int lane = gtid & 31, warp = gtid >> 5;
  const int lr = lane >> 2, lk = lane & 3;
  // tile slots of this warp: (ta[u], tb[u]), u < nt
  const int nt = warp < 2 ? 3 : 2;
  int ta[3], tb[3];
  ta[0] = warp == 0 ? 0 : warp == 1 ? 3 : warp == 2 ? 1 : 2;  tb[0] = warp == 0 ? 0 : warp == 1 ? 0 : warp == 2 ? 1 : 2;
  ta[1] = warp == 0 ? 0 : warp == 1 ? 3 : warp == 2 ? 1 : 3;  tb[1] = warp == 0 ? 1 : warp == 1 ? 1 : warp == 2 ? 2 : 3;
  ta[2] = warp == 0 ? 0 : 3;                                   tb[2] = 2;
  // complex products with three real tile products instead of four (3M): for conj(a) b
  //   T1 = ar br, T2 = ai bi, T3 = (ar - ai)(br + bi);  re = T1 + T2, im = T3 - T1 + T2
  // (normwise as accurate as the four-product form: every term is bounded by |a||b|)
  double t1[3][2], t2[3][2], t3[3][2];
#pragma unroll
  for (int u = 0; u < 3; ++u) { t1[u][0] = t1[u][1] = 0.0; t2[u][0] = t2[u][1] = 0.0; t3[u][0] = t3[u][1] = 0.0; }
  const int nch = (I.m + SV_R - 1) / SV_R;
#ifdef SV_TMA
  asm volatile("fence.proxy.async.shared::cta;\n" ::: "memory");   // ordinary writes to the ring (H, Qt of the last item) before bulk writes
  gsync(g);
#endif
#pragma unroll
  for (int p = 0; p < SV_NSTAGE - 1; ++p) {
#ifdef SV_TMA
    if (p < nch) load_chunk_tma(stages + p * SV_STAGE, SV_LDG, I, p * SV_R, I.m, gtid, RS, p);
#else
    if (p < nch) load_chunk(stages + p * SV_STAGE, SV_LDG, L, p * SV_R, I.m, gtid);
    cp_async_commit();
#endif
  }
  for (int c = 0; c < nch; ++c) {
#ifdef SV_TMA
    mbar_wait(RS.bar + c % SV_NSTAGE, (RS.phase >> (c % SV_NSTAGE)) & 1u);
    RS.phase ^= 1u << (c % SV_NSTAGE);
    gsync(g);  // everybody is done with chunk c - 1 (and sees the zero fill of chunk c): its stage may be refilled
    if (c + SV_NSTAGE - 1 < nch)
      load_chunk_tma(stages + ((c + SV_NSTAGE - 1) % SV_NSTAGE) * SV_STAGE, SV_LDG, I, (c + SV_NSTAGE - 1) * SV_R, I.m, gtid, RS, (c + SV_NSTAGE - 1) % SV_NSTAGE);
#else
    cp_async_wait<SV_NSTAGE - 2>();
    gsync(g);  // chunk c has landed for everybody, and everybody is done with chunk c - 1: its stage may be refilled
    if (c + SV_NSTAGE - 1 < nch)
      load_chunk(stages + ((c + SV_NSTAGE - 1) % SV_NSTAGE) * SV_STAGE, SV_LDG, L, (c + SV_NSTAGE - 1) * SV_R, I.m, gtid);
    cp_async_commit();
#endif
    const cplx* st = stages + (c % SV_NSTAGE) * SV_STAGE + lr * SV_LDG + lk;
    const int rows = min(SV_R, I.m - c * SV_R);
    const int nk = (rows + 3) >> 2;
    const cplx* pa0 = st + 8 * ta[0] * SV_LDG;   // slots 0 and 2 (if any) share the A tile of slot 0 or 1
    const cplx* pa1 = st + 8 * ta[1] * SV_LDG;
    const cplx* pb0 = st + 8 * tb[0] * SV_LDG;
    const cplx* pb1 = st + 8 * tb[1] * SV_LDG;
    const cplx* pb2 = st + 8 * tb[2] * SV_LDG;
#pragma unroll 1
    for (int ks = 0; ks < nk; ++ks) {
      const cplx a0 = pa0[4 * ks], a1 = pa1[4 * ks], b0 = pb0[4 * ks], b1 = pb1[4 * ks];
      const double a0d = a0.x - a0.y, a1d = a1.x - a1.y;
      dmma(t1[0][0], t1[0][1], a0.x, b0.x); dmma(t2[0][0], t2[0][1], a0.y, b0.y); dmma(t3[0][0], t3[0][1], a0d, b0.x + b0.y);
      dmma(t1[1][0], t1[1][1], a1.x, b1.x); dmma(t2[1][0], t2[1][1], a1.y, b1.y); dmma(t3[1][0], t3[1][1], a1d, b1.x + b1.y);
      if (nt == 3) {  // warp-uniform; the A tile of slot 2 is that of slot 0
        const cplx b2 = pb2[4 * ks];
        dmma(t1[2][0], t1[2][1], a0.x, b2.x); dmma(t2[2][0], t2[2][1], a0.y, b2.y); dmma(t3[2][0], t3[2][1], a0d, b2.x + b2.y);
      }
    }
  }
  double cre[3][2], cim[3][2];
#pragma unroll
  for (int u = 0; u < 3; ++u)
#pragma unroll
    for (int t = 0; t < 2; ++t) { cre[u][t] = t1[u][t] + t2[u][t]; cim[u][t] = (t3[u][t] - t1[u][t]) + t2[u][t]; }
  cp_async_wait<0>();
  gsync(g);  // every warp is done with the stages: Hs (aliased onto the ring) may be written
#pragma unroll
  for (int u = 0; u < 3; ++u) {
    if (u < nt) {
#pragma unroll
      for (int t = 0; t < 2; ++t) {
        const int r = 8 * ta[u] + lr, cidx = 8 * tb[u] + 2 * lk + t;
        if (warp == 1) Hs[cidx * SV_HLD + r] = make_double2(cre[u][t], -cim[u][t]);   // tile (3, j) -> (j, 3)
        else Hs[r * SV_HLD + cidx] = make_double2(cre[u][t], cim[u][t]);
      }
    }
  }
  gsync(g);
  // only the upper triangle of H is used from here on (the quick test and the EVD read row <= column)
  if (gtid < SV_W) Hs[gtid * SV_HLD + gtid].y = 0.0;
  gsync(g);
}

__device__ __forceinline__ double rsqrt_approx(double x) { double y; asm("rsqrt.approx.ftz.f64 %0, %1;" : "=d"(y) : "d"(x)); return y; }
__device__ __forceinline__ double rcp_approx(double x) { double y; asm("rcp.approx.ftz.f64 %0, %1;" : "=d"(y) : "d"(x)); return y; }

// pivot k of round t of the round-robin tournament over np2 players (not ordered: consecutive k give consecutive
// indices, which keeps the shared-memory accesses of a quarter warp in distinct banks)
__device__ __forceinline__ void pivot(int t, int k, int np2, int* p, int* q) {
  const int m = np2 - 1;
  if (k == 0) { *p = t; *q = m; return; }
  int a = t + k, b = t - k + m;
  if (a >= m) a -= m;
  if (b >= m) b -= m;
  *p = a; *q = b;
}

// ---- phase 2: two-sided Jacobi EVD of the Hermitian H (2*hp x 2*hp, hp = 16 or 8 pivots per round), Qt (stored
// transposed) accumulates the rotations; both in place in shared memory.
// Round t of a sweep rotates the hp disjoint pivots (p_k, q_k) of the round-robin tournament.  Rotation of a pivot
// (p, q) (= a scalar one-sided rotation of columns p, q, whose Gram entries are a = h_pp, b = h_qq, g = h_pq):
//   zeta = (b - a) / (2|g|), t = sign(zeta) / (|zeta| + sqrt(1 + zeta^2)), tau = t g/|g|, cs = 1/sqrt(1 + |tau|^2),
//   s = cs tau,  R = [[cs, s], [-conj(s), cs]].
// tau comes from the ~20-bit MUFU reciprocal / rsqrt (it only has to shrink the off-diagonal entry; the iteration is
// self-correcting), cs is computed in full precision so that R is unitary to rounding whatever tau is.  Where the
// new norms would be out of order the two result columns are exchanged (de Rijk: the larger norm goes to the lower index).
// Work split of a round: thread k < hp computes rotation k and rewrites its own 2 x 2 pivot block (closed form);
// after the barrier every 2 x 2 unit (rows of pivot ki, columns of pivot kj, ki < kj) is read, rotated from both
// sides and written, together with its mirror image, by one thread (H stays exactly Hermitian); the Q units
// (two rows x the two columns of a pivot) likewise.  The pivots of a round come from a small shared-memory table of the
// modulus ordering (pairs with (i + j) mod 2hp == round), the same pipelined cyclic-by-rows ordering as the outer one.
#ifdef EVD_CLK
__device__ long long evd_clk[20];
#endif
struct Rot { double cs, sr, si; int flag; };
// H is kept as its upper triangle only (row <= column): entry (r, c) of the Hermitian matrix
__device__ __forceinline__ cplx ldH(const cplx* H, int r, int c) {
  const cplx v = H[min(r, c) * SV_HLD + max(r, c)];
  return make_double2(v.x, r <= c ? v.y : -v.y);
}
__device__ __forceinline__ void stH(cplx* H, int r, int c, cplx v) {
  H[min(r, c) * SV_HLD + max(r, c)] = make_double2(v.x, r <= c ? v.y : -v.y);
}   // flag: 0 idle, 1 rotate, 3 rotate and exchange
__device__ __forceinline__ Rot load_rot(const double4* Rm, int k) {
  const double4 v = Rm[k];
  Rot r; r.cs = v.x; r.sr = v.y; r.si = v.z; r.flag = (int)v.w;
  return r;
}
// [x y] <- [x y] R :  x' = cs x - conj(s) y,  y' = s x + cs y
__device__ __forceinline__ void rot_cols(cplx& x, cplx& y, const Rot& r) {
  const cplx xn = make_double2(fma(-r.sr, y.x, fma(-r.si, y.y, r.cs * x.x)), fma(-r.sr, y.y, fma(r.si, y.x, r.cs * x.y)));
  const cplx yn = make_double2(fma(r.sr, x.x, fma(-r.si, x.y, r.cs * y.x)), fma(r.sr, x.y, fma(r.si, x.x, r.cs * y.y)));
  x = xn; y = yn;
}
// [x; y] <- R^H [x; y] :  x' = cs x - s y,  y' = conj(s) x + cs y
__device__ __forceinline__ void rot_rows(cplx& x, cplx& y, const Rot& r) {
  const cplx xn = make_double2(fma(-r.sr, y.x, fma(r.si, y.y, r.cs * x.x)), fma(-r.sr, y.y, fma(-r.si, y.x, r.cs * x.y)));
  const cplx yn = make_double2(fma(r.sr, x.x, fma(r.si, x.y, r.cs * y.x)), fma(r.sr, x.y, fma(-r.si, x.x, r.cs * y.y)));
  x = xn; y = yn;
}
// Pivot k of the round with residue rho of the modulus ordering over n players (n even, n/2 slots): the pairs
// (i, j), i < j, with (i + j) mod n == rho.  For even rho two players stay unpaired: they fill the last slot as an
// idle pivot (returned with bit 7 of q set), so that every row and column of H belongs to exactly one slot.
__device__ __forceinline__ uchar2 mod_pivot(int rho, int k, int n) {
  const int na = (rho + 1) >> 1;                       // pairs with i + j == rho
  const int nb = max(((rho + n + 1) >> 1) - rho - 1, 0);  // pairs with i + j == rho + n
  int p, q;
  if (k < na) { p = k; q = rho - k; }
  else if (k - na < nb) { p = rho + 1 + (k - na); q = rho + n - p; }
  else { p = rho >> 1; q = ((rho + n) >> 1) | 0x80; }
  return make_uchar2((unsigned char)p, (unsigned char)q);
}

__device__ __forceinline__ void evd_phase(cplx* H, cplx* Qt, double4* Rm, uchar2* tab, int hp, double tol2, int* inner, int inner_max, double quad, int g, int gtid) {
  const int tid = gtid;
  const int np2 = 2 * hp;
  for (int idx = tid; idx < np2 * hp; idx += SV_GROUP) tab[idx] = mod_pivot(idx / hp, idx % hp, np2);
  for (int idx = tid; idx < SV_W * SV_QLD; idx += SV_GROUP) {
    const int c = idx / SV_QLD, r = idx - c * SV_QLD;
    Qt[idx] = make_double2(r == c ? 1.0 : 0.0, 0.0);
  }
  // this thread's H unit: entry tid of the row-major list of the strict upper triangle ki < kj
  int uki = -1, ukj = 0;
  {
    int u = tid, ki = 0;
    if (u < hp * (hp - 1) / 2) {
      while (u >= hp - 1 - ki) { u -= hp - 1 - ki; ++ki; }
      uki = ki; ukj = ki + 1 + u;
    }
  }
  // Q units (two rows rp, rp + hp of Q x the two columns of pivot k) belong to warps 1..3 only: they are rotated one
  // round LATE, while warp 0 works out the rotations of the next round (Q does not enter the rotation angles)
  const int nqu = hp * hp;                       // 256 (or 64 for a single-panel item)
  int pend = 0, cur = 0;
  const uchar2* prow = tab;
  // Branch-free (an idle pivot carries the identity rotation cs = 1, s = 0, which leaves its operands bit-identical):
  // the loads, the arithmetic and the stores of a thread's up to three units (which never overlap) interleave freely.
  const int hsh = hp == U1_PB ? 4 : 3;            // hp = 1 << hsh
  int qk[3], qrp[3];                               // pivot and row pair of this thread's three Q units (-1: none, warp-uniform)
#pragma unroll
  for (int x = 0; x < 3; ++x) {
    const int u = tid - 32 + x * (SV_GROUP - 32);
    qk[x] = (tid >= 32 && u < nqu) ? u >> hsh : -1;
    qrp[x] = u & (hp - 1);
  }
  auto q_update = [&](const double4* Rp, const uchar2* rowp) {
#pragma unroll
    for (int x = 0; x < 3; ++x) {
      if (qk[x] >= 0) {   // warp-uniform
        const Rot rj = load_rot(Rp, qk[x]);
        const uchar2 vc = rowp[qk[x]];
        cplx* cp = Qt + vc.x * SV_QLD + qrp[x];
        cplx* cq = Qt + (vc.y & 0x7f) * SV_QLD + qrp[x];
        cplx q00 = cp[0], q01 = cq[0], q10 = cp[hp], q11 = cq[hp];
        rot_cols(q00, q01, rj); rot_cols(q10, q11, rj);
        cplx* dp = (rj.flag & 2) ? cq : cp;
        cplx* dq = (rj.flag & 2) ? cp : cq;
        dp[0] = q00; dq[0] = q01; dp[hp] = q10; dq[hp] = q11;
      }
    }
  };
  gsync(g);
#ifdef EVD_CLK   // probe build only (_work/evd_bench.cu): cycles of the segments of a round, per warp
  long long ck[5] = {0, 0, 0, 0, 0}, ct = clock64();
#define EVD_TICK(k) do { const long long _n = clock64(); ck[k] += _n - ct; ct = _n; } while (0)
#else
#define EVD_TICK(k) do {} while (0)
#endif
  for (int sw = 0; sw < inner_max; ++sw) {
    double mymax = 0.0;
    int sweep_any = 0;
    for (int t = 0; t < np2; ++t) {
      const uchar2* row = tab + ((t + 1) & (np2 - 1)) * hp;   // pivots of this round
      double4* Rc = Rm + cur * U1_PB;
      EVD_TICK(4);
      int rot = 0;
      if (tid < hp) {
        const uchar2 pv = row[tid];
        const int p = pv.x, q = pv.y & 0x7f;
        const double a = H[p * SV_HLD + p].x, b = H[q * SV_HLD + q].x;
        const cplx gg = ldH(H, p, q);
        const double g2 = fma(gg.x, gg.x, gg.y * gg.y), ab = a * b;
        double4 out = make_double4(1.0, 0.0, 0.0, 0.0);
        if (!(pv.y & 0x80) && ab > 0.0 && g2 > tol2 * ab && g2 > 1e-290) {
          rot = 1;
          mymax = fmax(mymax, g2 * rcp_approx(ab));
          // The rotation only has to shrink the off-diagonal entry (the iteration is self-correcting), so its angle is
          // worked out in SINGLE precision - short latencies, and not on the FP64 pipe the DMMA streams of the other CTAs
          // keep busy.  With d = (b - a)/2 and r = sqrt(d^2 + |g|^2) the small-angle Jacobi rotation has
          //   cos^2 = 1/2 + |d|/(2r),   s = sign(d) g / (2 r cos)      (t = sign(zeta)/(|zeta| + sqrt(1 + zeta^2)), zeta = d/|g|)
          // two MUFU rsqrt and a few FP32 operations.  g and d are first scaled by the power of two that brings the larger
          // component of g to [1, 2) (exact).  Where |d| > 1e15 |g| (d^2 would leave the single-precision range) the
          // small-angle limit cos = 1, s = g / (b - a) is exact to 1e-30.
          const int ex = (__double2hiint(gg.x) >> 20) & 0x7ff, ey = (__double2hiint(gg.y) >> 20) & 0x7ff;
          const double sc = __hiloint2double((2046 - min(max(ex, ey), 2045)) << 20, 0);
          const float gxf = (float)(gg.x * sc), gyf = (float)(gg.y * sc);
          const float dh = (float)((b - a) * (0.5 * sc));
          double c0, s0x, s0y;
          if (fabsf(dh) <= 1e15f) {
            const float ir = rsqrtf(fmaf(dh, dh, fmaf(gxf, gxf, gyf * gyf)));
            const float c2f = fmaf(0.5f * fabsf(dh), ir, 0.5f);
            const float icf = rsqrtf(c2f);
            const float kf = copysignf(0.5f * ir * icf, dh);
            c0 = (double)(c2f * icf); s0x = (double)(kf * gxf); s0y = (double)(kf * gyf);
          } else {
            const double ri = rcp_approx(b - a);
            c0 = 1.0; s0x = gg.x * ri; s0y = gg.y * ri;
          }
          // (cs, s) normalised in full precision: the rotation is unitary to rounding whatever the single-precision angle
          // is.  c^2 + |s|^2 = 1 + O(1e-6), so two Newton steps from 1 give 1/sqrt to ~1e-24.
          const double n2 = fma(c0, c0, fma(s0x, s0x, s0y * s0y));
          double y = fma(-0.5, n2, 1.5);
          y = y * fma(-0.5 * n2, y * y, 1.5);
          const double cs = c0 * y, sr = s0x * y, si = s0y * y;
          // the pivot block after the rotation, in closed form (x' = cs x - conj(s) y, y' = s x + cs y):
          //   a' = cs^2 a + |s|^2 b - 2 cs Re(conj(s) g),  b' = |s|^2 a + cs^2 b + 2 cs Re(conj(s) g),
          //   g' = x'^H y' = cs s (a - b) + cs^2 g - s^2 conj(g)
          const double s2 = sr * sr + si * si, c2 = cs * cs;
          const double cr = 2.0 * cs * (sr * gg.x + si * gg.y);
          const double an = fma(c2, a, fma(s2, b, -cr)), bn = fma(s2, a, fma(c2, b, cr));
          const double s2r = sr * sr - si * si, s2i = 2.0 * sr * si;   // s^2
          const double gnx = fma(cs * sr, a - b, fma(c2, gg.x, -(s2r * gg.x + s2i * gg.y)));
          const double gny = fma(cs * si, a - b, fma(c2, gg.y, -(s2i * gg.x - s2r * gg.y)));
          const bool swp = (p < q) ? (an < bn) : (bn < an);
          out = make_double4(cs, sr, si, swp ? 3.0 : 1.0);
          H[p * SV_HLD + p] = make_double2(swp ? bn : an, 0.0); H[q * SV_HLD + q] = make_double2(swp ? an : bn, 0.0);
          stH(H, p, q, make_double2(gnx, swp ? -gny : gny));
        }
        Rc[tid] = out;
      }
      EVD_TICK(0);
      // ... while warps 1..3 catch up on Q with the rotations of the previous round
      if (pend && tid >= 32) q_update(Rm + (cur ^ 1) * U1_PB, prow);
      // this thread's H unit is loaded before the barrier (the rotation threads only rewrite their own pivot blocks,
      // never an off-diagonal unit)
      int pi = 0, qi = 0, pj = 0, qj = 0;
      cplx b00, b01, b10, b11;
      if (uki >= 0) {
        const uchar2 vi = row[uki], vj = row[ukj];
        pi = vi.x; qi = vi.y & 0x7f; pj = vj.x; qj = vj.y & 0x7f;
        b00 = ldH(H, pi, pj); b01 = ldH(H, pi, qj); b10 = ldH(H, qi, pj); b11 = ldH(H, qi, qj);
      }
      EVD_TICK(1);
      const int any = gsync_or(g, rot);
      EVD_TICK(2);
      pend = any; prow = row; cur ^= 1;
      if (any) {  // uniform
        sweep_any = 1;
        if (uki >= 0) {
          // branch-free: an idle pivot carries the identity rotation, which leaves the unit bit-identical
          const Rot ri = load_rot(Rc, uki), rj = load_rot(Rc, ukj);
          rot_cols(b00, b01, rj); rot_cols(b10, b11, rj);
          rot_rows(b00, b10, ri); rot_rows(b01, b11, ri);
          // exchanges are applied to the destinations
          const int dpi = (ri.flag & 2) ? qi : pi, dqi = (ri.flag & 2) ? pi : qi;
          const int dpj = (rj.flag & 2) ? qj : pj, dqj = (rj.flag & 2) ? pj : qj;
          stH(H, dpi, dpj, b00); stH(H, dpi, dqj, b01); stH(H, dqi, dpj, b10); stH(H, dqi, dqj, b11);
        }
        EVD_TICK(3);
        gsync(g);
      }
    }
    if (!sweep_any) break;
    ++*inner;
    if (!gsync_or(g, mymax > quad)) break;
  }
  if (pend && tid >= 32) q_update(Rm + (cur ^ 1) * U1_PB, prow);
  gsync(g);
#ifdef EVD_CLK
  if ((tid & 31) == 0) for (int k = 0; k < 5; ++k) atomicAdd((unsigned long long*)&evd_clk[(tid >> 5) * 5 + k], (unsigned long long)ck[k]);
#endif
}

// ---- phase 3: [Pa Pb] <- [Pa Pb] Q over all mt rows.  Warp w owns tile column w (8 columns) and all row tiles
// of each 32-row chunk; its 32 x 8 slice of Q lives in registers as 8 B fragments.
__device__ __forceinline__ void update_phase(cplx* stages, const cplx* Qt, const Item& I, const Loader& L, RingState& RS, int g, int gtid) {
  const int lane = gtid & 31, warp = gtid >> 5;
  const int tj = warp;
  const int lr = lane >> 2, lk = lane & 3;
  // 3M complex products: T1 = ar br, T2 = ai bi, T3 = (ar + ai)(br + bi);  re = T1 - T2, im = T3 - T1 - T2
  double bre[8], bim[8], bsm[8];
#pragma unroll
  for (int ks = 0; ks < 8; ++ks) {
    const cplx v = Qt[(8 * tj + lr) * SV_QLD + 4 * ks + lk];   // Q[k][j], k = 4 ks + lk, j = 8 tj + lr
    bre[ks] = v.x; bim[ks] = v.y; bsm[ks] = v.x + v.y;
  }
#ifdef SV_TMA
  asm volatile("fence.proxy.async.shared::cta;\n" ::: "memory");
#endif
  gsync(g);  // Q (aliased onto the ring) is in registers everywhere: the ring may be refilled
  // the two output columns of this lane
  long long gcol[2]; bool cok[2];
#pragma unroll
  for (int t = 0; t < 2; ++t) {
    const int j = 8 * tj + 2 * lk + t;
    cok[t] = j < U1_PB ? j < I.na : j - U1_PB < I.nb;
    gcol[t] = (long long)I.col[j] * I.mt;
  }
  const int nch = (I.mt + SV_R - 1) / SV_R;
#pragma unroll
  for (int p = 0; p < SV_NSTAGE - 1; ++p) {
#ifdef SV_TMA
    if (p < nch) load_chunk_tma(stages + p * SV_STAGE, SV_LDU, I, p * SV_R, I.mt, gtid, RS, p);
#else
    if (p < nch) load_chunk(stages + p * SV_STAGE, SV_LDU, L, p * SV_R, I.mt, gtid);
    cp_async_commit();
#endif
  }
  for (int c = 0; c < nch; ++c) {
#ifdef SV_TMA
    mbar_wait(RS.bar + c % SV_NSTAGE, (RS.phase >> (c % SV_NSTAGE)) & 1u);
    RS.phase ^= 1u << (c % SV_NSTAGE);
    gsync(g);  // everybody is done with chunk c - 1 (and sees the zero fill of chunk c): its stage may be refilled
    if (c + SV_NSTAGE - 1 < nch)
      load_chunk_tma(stages + ((c + SV_NSTAGE - 1) % SV_NSTAGE) * SV_STAGE, SV_LDU, I, (c + SV_NSTAGE - 1) * SV_R, I.mt, gtid, RS, (c + SV_NSTAGE - 1) % SV_NSTAGE);
#else
    cp_async_wait<SV_NSTAGE - 2>();
    gsync(g);  // chunk c has landed for everybody, and everybody is done with chunk c - 1: its stage may be refilled
    if (c + SV_NSTAGE - 1 < nch)
      load_chunk(stages + ((c + SV_NSTAGE - 1) % SV_NSTAGE) * SV_STAGE, SV_LDU, L, (c + SV_NSTAGE - 1) * SV_R, I.mt, gtid);
    cp_async_commit();
#endif
    const cplx* st = stages + (c % SV_NSTAGE) * SV_STAGE;
    const int row0 = c * SV_R;
    const int rows = min(SV_R, I.mt - row0);
#pragma unroll
    for (int rt = 0; rt < SV_R / 8; ++rt) {
      if (8 * rt >= rows) break;
      double u1[2] = {0.0, 0.0}, u2[2] = {0.0, 0.0}, u3[2] = {0.0, 0.0};
      const cplx* pa = st + lk * SV_LDU + 8 * rt + lr;
#pragma unroll
      for (int ks = 0; ks < 8; ++ks) {
        const cplx a = pa[4 * ks * SV_LDU];
        dmma(u1[0], u1[1], a.x, bre[ks]); dmma(u2[0], u2[1], a.y, bim[ks]); dmma(u3[0], u3[1], a.x + a.y, bsm[ks]);
      }
      const int r = row0 + 8 * rt + lr;
      if (r < I.mt) {
        if (cok[0]) I.W[gcol[0] + r] = make_double2(u1[0] - u2[0], (u3[0] - u1[0]) - u2[0]);
        if (cok[1]) I.W[gcol[1] + r] = make_double2(u1[1] - u2[1], (u3[1] - u1[1]) - u2[1]);
      }
    }
  }
  cp_async_wait<0>();
  gsync(g);
}

// A sector of at most two panels (n <= 32) is a single item - all its columns - and depends on nothing: in a launch
// that consists of such sectors only (tiny bonds: the first layers of every trajectory, BASELINE.json's config 1) the CTA
// that draws a sector's ticket of round 0 iterates it to convergence on the spot: Gram - EVD run to convergence -
// update, until a visit finds nothing to rotate or only rotations in the quadratic regime.  Returns the visits made,
// negative if the limit was hit.  (A kernel of its own, svd_solo_kernel, launched in front of svd_kernel: it returns at
// once unless the launch consists of such sectors only, and svd_kernel then finds every sector finished.)
__device__ __forceinline__ int solo_sector(const Plan& P, int e, cplx* stages, cplx* Hs, cplx* Qs, double4* Rm, uchar2* tab, int* s_col,
                                        int inner_max, int R, RingState& RS) {
  const int gtid = threadIdx.x, g = 0;
  Item I;
  const int r = P.rows[e], q = P.cols[e], n = min(r, q);
  I.m = max(r, q);
  I.mt = I.m + n;
  I.W = P.W + P.goff[e];
  I.ca = 0; I.na = min(U1_PB, n);
  I.cb = U1_PB; I.nb = max(0, min(U1_PB, n - U1_PB));
  const double tol = SV_TOLFAC * 1.1102230246251565e-16 * sqrt((double)I.m);
  I.tol2 = tol * tol;
  if (gtid < SV_W) {
    const int j = gtid;
    const bool ok = j < U1_PB ? j < I.na : j - U1_PB < I.nb;
    s_col[j] = ok ? P.perm[P.svoff[e] + j] : 0;
  }
  I.col = s_col;
  gsync(g);
  const Loader L = make_loader(I, gtid);
  for (int iter = 0; iter < U1_MAXSWEEP; ++iter) {
    gram_phase(stages, Hs, I, L, RS, g, gtid);
    int todo = 0, big = 0;
    for (int idx = gtid; idx < SV_W * SV_W; idx += SV_GROUP) {
      const int p = idx >> 5, qq = idx & 31;
      if (p < qq) {
        const double a = Hs[p * SV_HLD + p].x, b = Hs[qq * SV_HLD + qq].x;
        const cplx gg = Hs[p * SV_HLD + qq];
        const double ab = a * b, g2 = gg.x * gg.x + gg.y * gg.y;
        if (ab > 0.0 && g2 > 1e-290) {
          todo |= (g2 > I.tol2 * ab) ? 1 : 0;
          big |= (g2 > SV_LASTPASS * ab) ? 1 : 0;
        }
      }
    }
    todo = gsync_or(g, todo);
    big = gsync_or(g, big);
    __syncthreads();
    if (!todo) return iter + 1;
    int inner = 0;
    evd_phase(Hs, Qs, Rm, tab, I.nb > 0 ? U1_PB : U1_PB / 2, I.tol2, &inner, inner_max + 4, 0.0, g, gtid);
    __syncthreads();
    update_phase(stages, Qs, I, L, RS, g, gtid);
    __syncthreads();   // the update's stores are visible to the CTA's next Gram pass
    if (gtid == 0) {
      const int sw = min(iter, U1_MAXSWEEP - 1);
      long long t1; asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(t1));
      atomicMax(&P.trace[1 + sw], t1);
      atomicAdd((unsigned long long*)&P.trace[1 + U1_MAXSWEEP + sw], 1ull);
      atomicAdd((unsigned long long*)&P.trace[1 + 2 * U1_MAXSWEEP + sw], (unsigned long long)inner);
    }
    if (!big) return iter + 1;
  }
  return -1;
}

__device__ __forceinline__ int ld_acquire(const int* p) {
  int v;
  asm volatile("ld.acquire.gpu.global.s32 %0, [%1];" : "=r"(v) : "l"(p) : "memory");
  return v;
}
#define SV_SPIN_LIMIT (1u << 24)   // x >= 100 ns: a dependency that does not resolve within seconds is reported, not waited for

// Work queue without grid-wide barriers.  Ticket T is item T % npair of round T / npair (the planner's list: the
// (np + 1) / 2 pair slots of every sector, longest sectors first).  An item of round t may start once all items of ITS
// sector of round t - 1 are done (a per-sector completion counter, release/acquire); items of different sectors never
// wait for each other, so every sector advances at its own pace and no CTA idles at a barrier.  Tickets are handed out
// in order and an item only waits for smaller tickets, whose holders are resident (cooperative launch): no deadlock.
__global__ void __launch_bounds__(U1_SVD_THREADS, SV_CTAS) svd_kernel(DevState S, Plan P, int G, int inner_max, int sms) {
  extern __shared__ __align__(16) unsigned char smraw[];
  __shared__ unsigned long long s_ticket;
  __shared__ int s_go, s_fin, s_rank;
  __shared__ int s_col[SV_W];
  const int tid = threadIdx.x, g = 0, gtid = tid;
  cplx* stages = reinterpret_cast<cplx*>(smraw);
  cplx* Hs = stages;                               // [32*33], aliased onto the ring (idle during the EVD)
  cplx* Qs = Hs + SV_W * SV_HLD;                   // [32*36], transposed
  double4* Rm = reinterpret_cast<double4*>(Qs + SV_W * SV_QLD);   // [2][16] rotations of the current and the previous EVD round
  uchar2* tab = reinterpret_cast<uchar2*>(Rm + 2 * U1_PB);         // [32][16] pivots of the modulus ordering
  const int nblk = P.cnt[0], npair = P.cnt[1], maxP = P.cnt[3];
  RingState RS;
#ifdef SV_TMA
  __shared__ __align__(8) unsigned long long s_bar[SV_NSTAGE];
  if (threadIdx.x == 0) {
    for (int i = 0; i < SV_NSTAGE; ++i) mbar_init(&s_bar[i], 1);
    asm volatile("fence.mbarrier_init.release.cluster;\n" ::: "memory");
  }
  RS.bar = s_bar; RS.phase = 0;
  __syncthreads();
#endif
  const int R = max(maxP, 1);                      // rounds of one cycle of the largest sector (= a "sweep" of the trace)
  const int E = G * S.NC;
  int* last_rot = P.flags;                         // [E] round after the last rotation outside the quadratic regime
  int* done_at = P.flags + E;                      // [E] round at which the sector was found converged (INT_MAX: not yet)
  int* done_cnt = P.flags + 2 * E;                 // [E] items of the sector completed so far, over all rounds
  // sched: [0..1] ticket (64 bit), [2] sectors finished, [3] CTAs that have left, [4] last round at which a sector finished,
  // [5] abort, [8 + smid] CTA ranks.
  // Load-dependent throttle: only as many CTAs per SM take items as the work warrants (the CTAs of an SM share the FP64
  // pipe, the shared-memory pipe and the issue slots: with few items per round every resident CTA beyond what is needed
  // only slows the others down; measured in profiles/r2_svd_tuning.md).
  int* sched = P.sched;
  if (tid == 0) { unsigned smid; asm volatile("mov.u32 %0, %%smid;" : "=r"(smid)); s_rank = atomicAdd(&sched[8 + (smid & 255)], 1); }
  __syncthreads();
  const int kact = min(SV_CTAS, max(SV_MIN_ACTIVE, (npair + SV_ITEMS_PER_CTA * sms - 1) / (SV_ITEMS_PER_CTA * sms)));
  if (blockIdx.x == 0 && tid == 0) { long long t0; asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(t0)); P.trace[0] = t0; }
#ifdef SV_PROFILE   // debug build only: clock64 per phase, summed over the grid into the tail of the trace
  long long pc[6] = {0, 0, 0, 0, 0, 0}, pt = clock64();
#define SV_TICK(k) do { const long long _n = clock64(); pc[k] += _n - pt; pt = _n; } while (0)
#else
#define SV_TICK(k) do {} while (0)
#endif
  const unsigned long long total = (unsigned long long)npair * (unsigned long long)(U1_MAXSWEEP * R);
  if (s_rank < kact && nblk > 0) {
    for (;;) {
      __syncthreads();
      if (tid == 0) {
        s_ticket = atomicAdd(reinterpret_cast<unsigned long long*>(sched), 1ull);
        s_go = (ld_acquire(&sched[2]) < nblk && ld_acquire(&sched[5]) == 0) ? 1 : 0;
      }
      __syncthreads();
      const unsigned long long T = s_ticket;
      if (T >= total || !s_go) break;
      const int tg = (int)(T / (unsigned long long)npair);
      const int it = (int)(T - (unsigned long long)tg * (unsigned long long)npair);
      Item I;
      const int e = P.pitem_e[it], k = P.pitem_k[it];
      const int r = P.rows[e], q = P.cols[e], n = min(r, q);
      I.m = max(r, q);
      I.mt = I.m + n;
      const int np = u1_ceil_div(n, U1_PB), slots = (np + 1) / 2;
      // Thread 0 takes the scheduling decisions for the CTA (every value it reads may change under its eyes):
      // s_go = 2: the sector was found finished in an earlier round - nothing to do (the item is still counted, so that
      //           nobody waits for it); 1: go; 0: abort.  s_fin: the sector is finished as of this round.
      SV_TICK(0);
      if (tid == 0) {
        int go = 1, fin = 0;
        if (ld_acquire(&done_at[e]) < tg) {
          go = 2;
        } else {
          // wait for the sector's items of the previous round
          const int need = tg * slots;
          unsigned spins = 0;
          while (ld_acquire(&done_cnt[e]) < need) {
            __nanosleep(100);
            if (++spins > SV_SPIN_LIMIT || ld_acquire(&sched[5]) != 0) { go = 0; break; }
          }
          if (!go) { atomicExch(&sched[5], 1); atomicExch(S.err, U1_ERR_SCHED); }
          // the sector is finished once np consecutive rounds (= every panel pair once) needed no rotation outside the
          // quadratic regime (last_rot is final for the rounds before tg: they are complete; a stamp of this very
          // round, tg + 1, reads as "not finished")
          else if (tg - ld_acquire(&last_rot[e]) >= np) {
            fin = 1;
            if (k == 0 && atomicMin(&done_at[e], tg) == 0x7fffffff) {
              atomicMax(&sched[4], tg);
              __threadfence();
              atomicAdd(&sched[2], 1);
            }
          }
        }
        if (go == 2) atomicAdd(&done_cnt[e], 1);
        s_go = go; s_fin = fin;
      }
      __syncthreads();
      if (s_go == 0) break;
      if (s_go == 2) continue;
      SV_TICK(4);
      bool have = !s_fin;
      // modulus ordering (a pipelined cyclic-by-rows ordering): round tg pairs the panels with (i + j) mod np == rho
      int pa = 0, pb = 1;
      if (np > 1) {
        const int rho = (tg + 1) % np;
        const int na = (rho + 1) >> 1;
        if (k < na) { pa = k; pb = rho - k; }
        else { pa = rho + 1 + (k - na); pb = rho + np - pa; }
        if (pa >= pb) have = false;
      }
      I.W = P.W + P.goff[e];
      I.ca = pa * U1_PB; I.na = min(U1_PB, n - I.ca);
      I.cb = pb * U1_PB; I.nb = pb < np ? min(U1_PB, n - I.cb) : 0;
      const double tol = SV_TOLFAC * 1.1102230246251565e-16 * sqrt((double)I.m);
      I.tol2 = tol * tol;
      int todo = 0, big = 0;
      Loader L;
      if (have) {
        // logical -> physical columns: the order of the initial column norms (descending), so that the sweeps start
        // from a sorted matrix; the rotations keep exchanging logical columns, the map itself never changes
        if (gtid < SV_W) {
          const int j = gtid;
          const bool ok = j < U1_PB ? j < I.na : j - U1_PB < I.nb;
          s_col[j] = ok ? P.perm[P.svoff[e] + (j < U1_PB ? I.ca + j : I.cb + j - U1_PB)] : 0;
        }
        I.col = s_col;
        gsync(g);
        SV_TICK(0);
        L = make_loader(I, gtid);
        gram_phase(stages, Hs, I, L, RS, g, gtid);
        SV_TICK(1);
        // quick test, same entries and arithmetic as the rotations: anything to do?
        for (int idx = gtid; idx < SV_W * SV_W; idx += SV_GROUP) {
          const int p = idx >> 5, qq = idx & 31;
          if (p < qq) {
            const double a = Hs[p * SV_HLD + p].x, b = Hs[qq * SV_HLD + qq].x;
            const cplx gg = Hs[p * SV_HLD + qq];
            const double ab = a * b, g2 = gg.x * gg.x + gg.y * gg.y;
            if (ab > 0.0 && g2 > 1e-290) {
              todo |= (g2 > I.tol2 * ab) ? 1 : 0;
              big |= (g2 > SV_LASTPASS * ab) ? 1 : 0;
            }
          }
        }
        todo = gsync_or(g, todo);
        big = gsync_or(g, big);
        // below SV_LASTPASS this visit's rotations leave relative off-diagonals of order 1e-6 sqrt(SV_LASTPASS) +
        // SV_LASTPASS << tol: such a visit does not restart the sector's count of clean rounds
        if (big && gtid == 0) atomicMax(&last_rot[e], tg + 1);
      }
      __syncthreads();
      SV_TICK(0);
      int inner = 0;
      if (todo) evd_phase(Hs, Qs, Rm, tab, I.nb > 0 ? U1_PB : U1_PB / 2, I.tol2, &inner, inner_max, SV_QUAD, g, gtid);
      __syncthreads();
      SV_TICK(2);
      if (todo) update_phase(stages, Qs, I, L, RS, g, gtid);
      SV_TICK(3);
      // done: publish (the update's stores and the stamp before the counter)
      __syncthreads();
      if (tid == 0) {
        if (todo) {  // trace of this launch (u1mps_svd_trace), one entry per R rounds
          const int sw = min(tg / R, U1_MAXSWEEP - 1);
          long long t1; asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(t1));
          atomicMax(&P.trace[1 + sw], t1);
          atomicAdd((unsigned long long*)&P.trace[1 + U1_MAXSWEEP + sw], 1ull);
          atomicAdd((unsigned long long*)&P.trace[1 + 2 * U1_MAXSWEEP + sw], (unsigned long long)inner);
        }
        __threadfence();
        atomicAdd(&done_cnt[e], 1);
      }
    }
  }
  SV_TICK(0);
#ifdef SV_PROFILE
  if (tid == 0) for (int k = 0; k < 5; ++k) atomicAdd((unsigned long long*)&P.trace[1 + 3 * U1_MAXSWEEP + 20 + k], (unsigned long long)pc[k]);
#endif
  // the last CTA to leave writes the statistics of the launch
  __syncthreads();
  if (tid == 0) { __threadfence(); s_go = (atomicAdd(&sched[3], 1) == (int)gridDim.x - 1) ? 1 : 0; }
  __syncthreads();
  if (s_go && nblk > 0) {
    __threadfence();
    const int fin = ld_acquire(&sched[2]);
    const int rounds = fin == nblk ? ld_acquire(&sched[4]) + 1 : U1_MAXSWEEP * R;
    const int nsw = min((rounds + R - 1) / R, U1_MAXSWEEP);
#ifndef SV_PROFILE
    // sectors not yet converged at the end of each sweep
    for (int bi = tid; bi < nblk; bi += U1_SVD_THREADS) {
      const int d = __ldcg(&done_at[P.blk[bi]]);
      for (int sw = 0; sw < nsw; ++sw)
        if (d > (sw + 1) * R - 1) atomicAdd((unsigned long long*)&P.trace[1 + 3 * U1_MAXSWEEP + sw], 1ull);
    }
#endif
    if (tid == 0) {
      atomicMax(&S.err[1], nsw);
      if (fin < nblk && ld_acquire(&sched[5]) == 0) atomicAdd(&S.err[2], nblk - fin);
      // end time of every sweep: the latest completion of one of its rotating items (sectors advance at their own
      // pace, so sweeps overlap; a sweep without rotations ends with the launch), made monotone
      long long t1; asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(t1));
      long long prev = P.trace[0];
      for (int sw = 0; sw < nsw; ++sw) {
        long long v = P.trace[1 + sw];
        if (v == 0) v = t1;
        v = max(v, prev);
        P.trace[1 + sw] = v;
        prev = v;
      }
    }
  }
}

__global__ void __launch_bounds__(U1_SVD_THREADS, SV_CTAS) svd_solo_kernel(Plan P, int G, int NC, int inner_max) {
  extern __shared__ __align__(16) unsigned char smraw[];
  __shared__ int s_col[SV_W];
  const int nblk = P.cnt[0], maxP = P.cnt[3];
  if (maxP > 2 || nblk == 0) return;
  RingState RS;
#ifdef SV_TMA
  __shared__ __align__(8) unsigned long long s_bar[SV_NSTAGE];
  if (threadIdx.x == 0) {
    for (int i = 0; i < SV_NSTAGE; ++i) mbar_init(&s_bar[i], 1);
    asm volatile("fence.mbarrier_init.release.cluster;\n" ::: "memory");
  }
  RS.bar = s_bar; RS.phase = 0;
  __syncthreads();
#endif

  cplx* stages = reinterpret_cast<cplx*>(smraw);
  cplx* Hs = stages;
  cplx* Qs = Hs + SV_W * SV_HLD;
  double4* Rm = reinterpret_cast<double4*>(Qs + SV_W * SV_QLD);
  uchar2* tab = reinterpret_cast<uchar2*>(Rm + 2 * U1_PB);
  const int R = max(maxP, 1), E = G * NC;
  int* done_at = P.flags + E;
  for (int bi = blockIdx.x; bi < nblk; bi += gridDim.x) {
    const int e = P.blk[bi];
    __syncthreads();
    const int visits = solo_sector(P, e, stages, Hs, Qs, Rm, tab, s_col, inner_max, R, RS);
    __syncthreads();
    if (threadIdx.x == 0 && visits > 0) {   // (a sector that hit the limit stays unfinished: svd_kernel reports it)
      atomicMin(&done_at[e], visits * R - 1);
      atomicMax(&P.sched[4], visits * R - 1);
      __threadfence();
      atomicAdd(&P.sched[2], 1);
    }
  }
}

// sigma_j = norm of column j of G (top m rows), then sort each sector descending (ties: lower
// column first).  One CTA per sector; bitonic sort in shared memory (n <= 4096).
#define SORT_THREADS 1024
__global__ void __launch_bounds__(SORT_THREADS) sigma_sort_kernel(Plan P) {
  extern __shared__ __align__(16) unsigned char smraw[];
  double* key = reinterpret_cast<double*>(smraw);
  int* idx = reinterpret_cast<int*>(key + U1MPS_SORT_MAX);
  const int nblk = P.cnt[0];
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  for (int bi = blockIdx.x; bi < nblk; bi += gridDim.x) {
    const int e = P.blk[bi];
    const int r = P.rows[e], q = P.cols[e], m = max(r, q), n = min(r, q), mt = m + n;
    const cplx* W = P.W + P.goff[e];
    int n2 = 1;
    while (n2 < n) n2 <<= 1;
    __syncthreads();
    for (int j = warp; j < n; j += SORT_THREADS / 32) {
      const cplx* col = W + (long long)j * mt;
      double a = 0.0;
      for (int rr = lane; rr < m; rr += 32) { const cplx v = __ldcg(col + rr); a = fma(v.x, v.x, a); a = fma(v.y, v.y, a); }
      a = warp_sum(a);
      if (lane == 0) { key[j] = sqrt(a); idx[j] = j; P.sv[P.svoff[e] + j] = sqrt(a); }
    }
    for (int j = n + tid; j < n2; j += SORT_THREADS) { key[j] = -1.0; idx[j] = 0x7fffffff; }
    __syncthreads();
    for (int k = 2; k <= n2; k <<= 1)
      for (int jj = k >> 1; jj > 0; jj >>= 1) {
        for (int i = tid; i < n2; i += SORT_THREADS) {
          const int l = i ^ jj;
          if (l > i) {
            const double ki = key[i], kl = key[l];
            const int ii = idx[i], il = idx[l];
            const bool before = (ki > kl) || (ki == kl && ii < il);  // i should precede l in descending order
            const bool up = ((i & k) == 0);
            if (up ? !before : before) { key[i] = kl; key[l] = ki; idx[i] = il; idx[l] = ii; }
          }
        }
        __syncthreads();
      }
    for (int j = tid; j < n; j += SORT_THREADS) { P.svs[P.svoff[e] + j] = key[j]; P.perm[P.svoff[e] + j] = idx[j]; }
  }
}

cudaError_t u1_svd_configure(int* grid, int* smem_bytes, int sms) {
  const int smem = SV_SMEM_BYTES;
  cudaError_t err = cudaFuncSetAttribute(svd_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, smem);
  if (err != cudaSuccess) return err;
  err = cudaFuncSetAttribute(svd_solo_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, smem);
  if (err != cudaSuccess) return err;
  err = cudaFuncSetAttribute(sigma_sort_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, U1MPS_SORT_MAX * 12);
  if (err != cudaSuccess) return err;
  int occ = 0;
  err = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, svd_kernel, U1_SVD_THREADS, smem);
  if (err != cudaSuccess) return err;
  if (occ < 1) return cudaErrorLaunchOutOfResources;
  *grid = sms * occ;
  *smem_bytes = smem;
  return cudaSuccess;
}

cudaError_t u1_launch_svd(const DevState& S, const Plan& P, int G, const LaunchCfg& L) {
  DevState s = S; Plan p = P; int gcount = G;
  int inner_max = SV_INNER_MAX;
  int sms = L.sms;
  void* args[] = {&s, &p, &gcount, &inner_max, &sms};
  // column norms of Theta sorted descending -> P.perm: the logical column order of the Jacobi iteration
  L.prof->begin(U1_ST_SORT, L.stream);
  sigma_sort_kernel<<<L.sms * 2, SORT_THREADS, U1MPS_SORT_MAX * 12, L.stream>>>(P);
  L.prof->end(L.stream);
  int grid = L.svd_grid;
#ifdef SV_PROFILE   // debug build only: CTAs per SM from the environment (phase latencies without contention)
  if (getenv("SV_PROFILE_CTAS")) grid = L.sms * atoi(getenv("SV_PROFILE_CTAS"));
#endif
  L.prof->begin(U1_ST_SVD, L.stream);
  svd_solo_kernel<<<L.sms * 2, U1_SVD_THREADS, (size_t)L.svd_smem, L.stream>>>(P, G, S.NC, inner_max);
  cudaError_t err = cudaLaunchCooperativeKernel((void*)svd_kernel, dim3(grid), dim3(U1_SVD_THREADS), args,
                                                (size_t)L.svd_smem, L.stream);
  L.prof->end(L.stream);
  if (err != cudaSuccess) return err;
  L.prof->begin(U1_ST_SORT, L.stream);
  sigma_sort_kernel<<<L.sms * 2, SORT_THREADS, U1MPS_SORT_MAX * 12, L.stream>>>(P);
  L.prof->end(L.stream);
  *L.launches += 4;
  return cudaGetLastError();
}
