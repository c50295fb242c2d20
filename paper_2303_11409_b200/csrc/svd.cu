// svd.cu — step a3: one SVD per centre-charge sector ("Singular value decompositions are
// then performed on each Theta(c^[k])"; Eq.12), for all sectors of all gates of the chunk at once.
// The paper calls a library SVD (L131); here it is a batched one-sided (Hestenes) BLOCK Jacobi SVD:
// the columns of the stacked matrix [G; J] (G = Theta(c) or its conjugate transpose so that
// m >= n, J = identity) are made mutually orthogonal; then sigma_j = |G_j|, left vectors
// G_j / sigma_j, right vectors J_j.
//
// Blocking.  Columns are grouped in panels of U1_PB = 16.  A work item is a panel pair P = [Pa Pb]
// (32 columns):
//   1. Gram   H = P^H P over the m rows of G           (FP64 DMMA.8x8x4 tiles, chunks of 64 rows staged
//                                                        in shared memory by a 3-stage cp.async ring)
//   2. EVD    H = Q diag Q^H by two-sided Jacobi in shared memory (parallel round-robin ordering, 16
//             rotations per round, 16 x 16 two-by-two units, one per thread; rotations sort the pair by
//             norm, de Rijk style, which is what makes graded spectra converge)
//   3. update [Pa Pb] <- [Pa Pb] Q over all m + n rows  (DMMA again, Q held in registers as B fragments)
// A persistent cooperative grid walks the round-robin tournament of panel pairs of every sector in
// lock step (one grid sync per round, items handed out through an atomic ticket); convergence is
// decided on the device per sector (a sweep in which no item had an off-diagonal Gram entry above
// tol * sqrt(h_pp h_qq)), no host round trip.
#include <cooperative_groups.h>
#include "common.cuh"
namespace cg = cooperative_groups;

#define SV_W 32                      // columns of a pair item
#define SV_R 64                      // rows per staged chunk
#define SV_LDG 68                    // shared-memory leading dimension (complex elements) in the Gram phase: 4 mod 8
#define SV_LDU 66                    // ... in the update phase: 2 mod 8 (both: conflict-free LDS.128 fragment loads)
#define SV_STAGE (SV_W * SV_LDG)     // complex elements per stage
#define SV_NSTAGE 3
#define SV_HLD 33                    // leading dimension of the 32 x 32 Gram / eigenvector matrices
#define SV_INNER_MAX 3               // inner EVD sweeps per item (the outer iteration finishes the job)
#define SV_QUAD 1e-14                // stop the inner EVD after a sweep whose largest relative off-diagonal^2 was below this
#define SV_SMEM_BYTES (SV_NSTAGE * SV_STAGE * 16)

__device__ __forceinline__ double warp_sum(double v) {
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
  return v;
}

// D(8x8) += A(8x4, row) * B(4x8, col), FP64 tensor tile (SASS: DMMA.8x8x4).
// Fragments: a = A[lane>>2][lane&3], b = B[lane&3][lane>>2], c0/c1 = C[lane>>2][2*(lane&3) + 0/1].
__device__ __forceinline__ void dmma(double& c0, double& c1, double a, double b) {
  asm("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};\n" : "+d"(c0), "+d"(c1) : "d"(a), "d"(b));
}

__device__ __forceinline__ void cp_async16(void* smem, const void* gmem, int src_bytes) {
  const unsigned s = (unsigned)__cvta_generic_to_shared(smem);
  asm volatile("cp.async.cg.shared.global [%0], [%1], 16, %2;\n" ::"r"(s), "l"(gmem), "r"(src_bytes) : "memory");
}
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;\n" ::: "memory"); }
template <int N>
__device__ __forceinline__ void cp_async_wait() { asm volatile("cp.async.wait_group %0;\n" ::"n"(N) : "memory"); }

__device__ __forceinline__ cplx cmul(cplx a, cplx b) { return make_double2(a.x * b.x - a.y * b.y, a.x * b.y + a.y * b.x); }
__device__ __forceinline__ cplx cmulc(cplx a, cplx b) {  // conj(a) * b
  return make_double2(a.x * b.x + a.y * b.y, a.x * b.y - a.y * b.x);
}
__device__ __forceinline__ cplx cadd(cplx a, cplx b) { return make_double2(a.x + b.x, a.y + b.y); }

// circle-method round robin over np2 (even) players: slot k of round t -> (a, b), a < b
__device__ __forceinline__ void rr_pair(int t, int k, int np2, int* a, int* b) {
  const int q = np2 - 1;
  if (k == 0) { *a = t % q; *b = q; }
  else { *a = (t + k) % q; *b = (t - k + 2 * q) % q; }
  if (*a > *b) { int s = *a; *a = *b; *b = s; }
}

struct Item {
  cplx* W;        // stacked (m + n) x n column-major Jacobi matrix of the sector
  int m, mt;      // rows of G; m + n = leading dimension
  int ca, na;     // first column / number of columns of panel a
  int cb, nb;     // ... of panel b (nb = 0: single-panel item)
  double tol2;
};

// Stage rows [row0, row0 + 64) x the 32 columns of the item into shared memory (column-major, leading dimension ld);
// rows >= rowlim and absent columns are zero-filled.
__device__ __forceinline__ void load_chunk(cplx* st, int ld, const Item& I, int row0, int rowlim) {
  const int r = threadIdx.x & (SV_R - 1);
  const bool rok = row0 + r < rowlim;
#pragma unroll
  for (int it = 0; it < SV_W * SV_R / U1_SVD_THREADS; ++it) {
    const int j = (threadIdx.x >> 6) + it * (U1_SVD_THREADS / SV_R);
    const bool ok = rok && (j < U1_PB ? j < I.na : j - U1_PB < I.nb);
    const long long gcol = j < U1_PB ? I.ca + j : I.cb + j - U1_PB;
    const cplx* src = ok ? I.W + gcol * I.mt + row0 + r : I.W;
    cp_async16(st + j * ld + r, src, ok ? 16 : 0);
  }
}

// ---- phase 1: H = P^H P over rows [0, m).  Warp w owns tile row w/2 and tile columns 2(w%2), 2(w%2)+1 of the 4 x 4 tiles.
__device__ __forceinline__ void gram_phase(cplx* stages, cplx* Hs, const Item& I) {
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  const int ti = warp >> 1, tj = (warp & 1) * 2;
  const int lr = lane >> 2, lk = lane & 3;
  double cre[2][2] = {{0.0, 0.0}, {0.0, 0.0}}, cim[2][2] = {{0.0, 0.0}, {0.0, 0.0}};
  const int nch = (I.m + SV_R - 1) / SV_R;
  load_chunk(stages, SV_LDG, I, 0, I.m);
  cp_async_commit();
  if (nch > 1) load_chunk(stages + SV_STAGE, SV_LDG, I, SV_R, I.m);
  cp_async_commit();
  for (int c = 0; c < nch; ++c) {
    cp_async_wait<1>();
    __syncthreads();
    if (c + 2 < nch) load_chunk(stages + ((c + 2) % SV_NSTAGE) * SV_STAGE, SV_LDG, I, (c + 2) * SV_R, I.m);
    cp_async_commit();
    const cplx* st = stages + (c % SV_NSTAGE) * SV_STAGE;
    const int rows = min(SV_R, I.m - c * SV_R);
    const int nk = (rows + 3) >> 2;
    const cplx* pa = st + (8 * ti + lr) * SV_LDG + lk;
    const cplx* pb0 = st + (8 * tj + lr) * SV_LDG + lk;
    const cplx* pb1 = pb0 + 8 * SV_LDG;
#pragma unroll 4
    for (int ks = 0; ks < nk; ++ks) {
      const cplx a = pa[4 * ks], b0 = pb0[4 * ks], b1 = pb1[4 * ks];
      const double nai = -a.y;
      // conj(a) * b : re = ar br + ai bi ; im = ar bi - ai br
      dmma(cre[0][0], cre[0][1], a.x, b0.x); dmma(cre[0][0], cre[0][1], a.y, b0.y);
      dmma(cim[0][0], cim[0][1], a.x, b0.y); dmma(cim[0][0], cim[0][1], nai, b0.x);
      dmma(cre[1][0], cre[1][1], a.x, b1.x); dmma(cre[1][0], cre[1][1], a.y, b1.y);
      dmma(cim[1][0], cim[1][1], a.x, b1.y); dmma(cim[1][0], cim[1][1], nai, b1.x);
    }
  }
  cp_async_wait<0>();
  __syncthreads();  // every warp is done with the stages: Hs (aliased onto stages 1..2) may be written
#pragma unroll
  for (int u = 0; u < 2; ++u)
#pragma unroll
    for (int t = 0; t < 2; ++t)
      Hs[(8 * ti + lr) * SV_HLD + 8 * (tj + u) + 2 * lk + t] = make_double2(cre[u][t], cim[u][t]);
  __syncthreads();
  // exact Hermitian symmetry from the upper triangle (the quick test and the rotations read p < q only)
  for (int idx = threadIdx.x; idx < SV_W * SV_W; idx += U1_SVD_THREADS) {
    const int p = idx >> 5, q = idx & 31;
    if (p > q) { const cplx v = Hs[q * SV_HLD + p]; Hs[p * SV_HLD + q] = make_double2(v.x, -v.y); }
    else if (p == q) Hs[p * SV_HLD + p].y = 0.0;
  }
  __syncthreads();
}

// ---- phase 2: two-sided Jacobi EVD of the Hermitian H (2*hp x 2*hp, hp = 16 or 8 pairs per round), Q accumulates the
// rotations.  H and Q are double-buffered (Hs/Qs: [2][32*33]); returns the index of the buffer holding the result.
// Rotation of the pivot (p, q), p < q (same formulas as a scalar one-sided rotation of columns p, q, whose Gram
// entries are a = h_pp, b = h_qq, g = h_pq):  zeta = (b - a) / (2|g|), t = sign(zeta) / (|zeta| + sqrt(1 + zeta^2)),
// cs = 1/sqrt(1 + t^2), s = cs t g/|g|,  R = [[cs, s], [-conj(s), cs]]; if the new norms a - t|g| < b + t|g| the two
// columns of R are swapped so that the larger norm ends up in the lower column.
__device__ __forceinline__ int evd_phase(cplx* Hs, cplx* Qs, cplx (*Rm)[4], int* sp, int* sq, int hp, double tol2) {
  const int tid = threadIdx.x;
  const int np2 = 2 * hp;
  for (int idx = tid; idx < SV_W * SV_W; idx += U1_SVD_THREADS) {  // both buffers: a round rewrites only the 2hp x 2hp corner
    const int r = idx >> 5, c = idx & 31;
    const cplx one = make_double2(r == c ? 1.0 : 0.0, 0.0);
    Qs[r * SV_HLD + c] = one;
    Qs[SV_W * SV_HLD + r * SV_HLD + c] = one;
    Hs[SV_W * SV_HLD + r * SV_HLD + c] = Hs[r * SV_HLD + c];
  }
  int cur = 0;
  const int ki = tid / hp, kj = tid % hp;
  const bool worker = tid < hp * hp;
  __syncthreads();
  for (int sw = 0; sw < SV_INNER_MAX; ++sw) {
    double mymax = 0.0;
    int sweep_any = 0;
    for (int t = 0; t < np2 - 1; ++t) {
      int rot = 0;
      if (tid < hp) {
        int p, q;
        rr_pair(t, tid, np2, &p, &q);
        const cplx* H = Hs + cur * (SV_W * SV_HLD);
        const double a = H[p * SV_HLD + p].x, b = H[q * SV_HLD + q].x;
        const cplx g = H[p * SV_HLD + q];
        const double g2 = g.x * g.x + g.y * g.y, ab = a * b;
        cplx r00 = make_double2(1.0, 0.0), r01 = make_double2(0.0, 0.0), r10 = r01, r11 = r00;
        if (ab > 0.0 && g2 > tol2 * ab) {
          rot = 1;
          mymax = fmax(mymax, g2 / ab);
          const double ag = sqrt(g2);
          const double zeta = (b - a) / (2.0 * ag);
          const double tt = copysign(1.0, zeta) / (fabs(zeta) + sqrt(1.0 + zeta * zeta));
          const double cs = rsqrt(1.0 + tt * tt);
          const double sn = cs * tt;
          const double sr = sn * g.x / ag, si = sn * g.y / ag;
          if ((a - tt * ag) < (b + tt * ag)) {  // swapped columns
            r00 = make_double2(sr, si); r01 = make_double2(cs, 0.0);
            r10 = make_double2(cs, 0.0); r11 = make_double2(-sr, si);
          } else {
            r00 = make_double2(cs, 0.0); r01 = make_double2(sr, si);
            r10 = make_double2(-sr, si); r11 = make_double2(cs, 0.0);
          }
        }
        Rm[tid][0] = r00; Rm[tid][1] = r01; Rm[tid][2] = r10; Rm[tid][3] = r11;
        sp[tid] = p; sq[tid] = q;
      }
      const int any = __syncthreads_or(rot);
      if (!any) continue;  // nobody rotated: buffers stay as they are (uniform branch)
      sweep_any = 1;
      if (worker) {
        const cplx* H = Hs + cur * (SV_W * SV_HLD);
        cplx* Hn = Hs + (cur ^ 1) * (SV_W * SV_HLD);
        const cplx* Q = Qs + cur * (SV_W * SV_HLD);
        cplx* Qn = Qs + (cur ^ 1) * (SV_W * SV_HLD);
        const int pi = sp[ki], qi = sq[ki], pj = sp[kj], qj = sq[kj];
        const cplx j00 = Rm[kj][0], j01 = Rm[kj][1], j10 = Rm[kj][2], j11 = Rm[kj][3];
        const cplx i00 = Rm[ki][0], i01 = Rm[ki][1], i10 = Rm[ki][2], i11 = Rm[ki][3];
        const cplx b00 = H[pi * SV_HLD + pj], b01 = H[pi * SV_HLD + qj], b10 = H[qi * SV_HLD + pj], b11 = H[qi * SV_HLD + qj];
        // T = B Rj ; B' = Ri^H T
        const cplx t00 = cadd(cmul(b00, j00), cmul(b01, j10)), t01 = cadd(cmul(b00, j01), cmul(b01, j11));
        const cplx t10 = cadd(cmul(b10, j00), cmul(b11, j10)), t11 = cadd(cmul(b10, j01), cmul(b11, j11));
        Hn[pi * SV_HLD + pj] = cadd(cmulc(i00, t00), cmulc(i10, t10));
        Hn[pi * SV_HLD + qj] = cadd(cmulc(i00, t01), cmulc(i10, t11));
        Hn[qi * SV_HLD + pj] = cadd(cmulc(i01, t00), cmulc(i11, t10));
        Hn[qi * SV_HLD + qj] = cadd(cmulc(i01, t01), cmulc(i11, t11));
        // Q rows 2ki, 2ki+1, columns (pj, qj):  Q' = Q Rj
        const int r0 = 2 * ki, r1 = r0 + 1;
        const cplx q00 = Q[r0 * SV_HLD + pj], q01 = Q[r0 * SV_HLD + qj], q10 = Q[r1 * SV_HLD + pj], q11 = Q[r1 * SV_HLD + qj];
        Qn[r0 * SV_HLD + pj] = cadd(cmul(q00, j00), cmul(q01, j10));
        Qn[r0 * SV_HLD + qj] = cadd(cmul(q00, j01), cmul(q01, j11));
        Qn[r1 * SV_HLD + pj] = cadd(cmul(q10, j00), cmul(q11, j10));
        Qn[r1 * SV_HLD + qj] = cadd(cmul(q10, j01), cmul(q11, j11));
      }
      cur ^= 1;
      __syncthreads();
    }
    if (!sweep_any) break;
    if (!__syncthreads_or(mymax > SV_QUAD)) break;
  }
  return cur;
}

// ---- phase 3: [Pa Pb] <- [Pa Pb] Q over all mt rows.  Warp w owns tile column w%4 (8 columns) and the row tiles
// (w/4), (w/4)+2, ... of each 64-row chunk; its 32 x 8 slice of Q lives in registers as 8 B fragments.
__device__ __forceinline__ void update_phase(cplx* stages, const cplx* Q, const Item& I) {
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  const int tj = warp & 3, rh = warp >> 2;
  const int lr = lane >> 2, lk = lane & 3;
  double bre[8], bim[8];
#pragma unroll
  for (int ks = 0; ks < 8; ++ks) {
    const cplx v = Q[(4 * ks + lk) * SV_HLD + 8 * tj + lr];
    bre[ks] = v.x; bim[ks] = v.y;
  }
  __syncthreads();  // Q (aliased onto stages 1..2) is in registers everywhere: the ring may be refilled
  // the two output columns of this lane
  long long gcol[2]; bool cok[2];
#pragma unroll
  for (int t = 0; t < 2; ++t) {
    const int j = 8 * tj + 2 * lk + t;
    cok[t] = j < U1_PB ? j < I.na : j - U1_PB < I.nb;
    gcol[t] = (j < U1_PB ? I.ca + j : I.cb + j - U1_PB) * (long long)I.mt;
  }
  const int nch = (I.mt + SV_R - 1) / SV_R;
  load_chunk(stages, SV_LDU, I, 0, I.mt);
  cp_async_commit();
  if (nch > 1) load_chunk(stages + SV_STAGE, SV_LDU, I, SV_R, I.mt);
  cp_async_commit();
  for (int c = 0; c < nch; ++c) {
    cp_async_wait<1>();
    __syncthreads();
    if (c + 2 < nch) load_chunk(stages + ((c + 2) % SV_NSTAGE) * SV_STAGE, SV_LDU, I, (c + 2) * SV_R, I.mt);
    cp_async_commit();
    const cplx* st = stages + (c % SV_NSTAGE) * SV_STAGE;
    const int row0 = c * SV_R;
    const int rows = min(SV_R, I.mt - row0);
#pragma unroll
    for (int rt = rh; rt < SV_R / 8; rt += 2) {
      if (8 * rt >= rows) break;
      double cre[2] = {0.0, 0.0}, cim[2] = {0.0, 0.0};
      const cplx* pa = st + lk * SV_LDU + 8 * rt + lr;
#pragma unroll
      for (int ks = 0; ks < 8; ++ks) {
        const cplx a = pa[4 * ks * SV_LDU];
        const double nai = -a.y;
        // a * b : re = ar br - ai bi ; im = ar bi + ai br
        dmma(cre[0], cre[1], a.x, bre[ks]); dmma(cre[0], cre[1], nai, bim[ks]);
        dmma(cim[0], cim[1], a.x, bim[ks]); dmma(cim[0], cim[1], a.y, bre[ks]);
      }
      const int r = row0 + 8 * rt + lr;
      if (r < I.mt) {
        if (cok[0]) I.W[gcol[0] + r] = make_double2(cre[0], cim[0]);
        if (cok[1]) I.W[gcol[1] + r] = make_double2(cre[1], cim[1]);
      }
    }
  }
  cp_async_wait<0>();
  __syncthreads();
}

__global__ void __launch_bounds__(U1_SVD_THREADS, 2) svd_kernel(DevState S, Plan P) {
  extern __shared__ __align__(16) unsigned char smraw[];
  cplx* stages = reinterpret_cast<cplx*>(smraw);
  cplx* Hs = stages + SV_STAGE;                    // [2][32*33], aliased onto stages 1..2 (idle during the EVD)
  cplx* Qs = Hs + 2 * SV_W * SV_HLD;               // [2][32*33]
  __shared__ cplx Rm[U1_PB][4];
  __shared__ int sp[U1_PB], sq[U1_PB];
  __shared__ unsigned s_ticket;
  cg::grid_group grid = cg::this_grid();
  const int nblk = P.cnt[0], npair = P.cnt[1], maxP = P.cnt[3];
  const int rounds = max(maxP - 1, 1);
  const int tid = threadIdx.x;
  unsigned base = 0;
  unsigned* ticket = reinterpret_cast<unsigned*>(P.cnt + 6);
  int sweep = 0;
  for (; sweep < U1_MAXSWEEP && nblk > 0; ++sweep) {
    for (int t = 0; t < rounds; ++t) {
      for (;;) {
        __syncthreads();
        if (tid == 0) s_ticket = atomicAdd(ticket, 1u) - base;
        __syncthreads();
        const unsigned it = s_ticket;
        if (it >= (unsigned)npair) break;
        const int e = P.pitem_e[it], k = P.pitem_k[it];
        if (sweep > 0 && __ldcg(&P.flags[e * U1_MAXSWEEP + sweep - 1]) == 0) continue;  // sector converged
        const int r = P.rows[e], q = P.cols[e];
        Item I;
        I.m = max(r, q);
        const int n = min(r, q);
        I.mt = I.m + n;
        const int np = u1_ceil_div(n, U1_PB);
        const int np2 = np + (np & 1);
        if (t >= max(np2 - 1, 1)) continue;
        int pa, pb;
        rr_pair(t, k, max(np2, 2), &pa, &pb);
        if (pb >= np && np > 1) continue;  // bye (odd number of panels)
        I.W = P.W + P.goff[e];
        I.ca = pa * U1_PB; I.na = min(U1_PB, n - I.ca);
        I.cb = pb * U1_PB; I.nb = pb < np ? min(U1_PB, n - I.cb) : 0;
        const double tol = 8.0 * 1.1102230246251565e-16 * sqrt((double)I.m);
        I.tol2 = tol * tol;
        gram_phase(stages, Hs, I);
        // quick test, same entries and arithmetic as the rotations: anything to do?
        int todo = 0;
        for (int idx = tid; idx < SV_W * SV_W; idx += U1_SVD_THREADS) {
          const int p = idx >> 5, qq = idx & 31;
          if (p < qq) {
            const double a = Hs[p * SV_HLD + p].x, b = Hs[qq * SV_HLD + qq].x;
            const cplx g = Hs[p * SV_HLD + qq];
            const double ab = a * b;
            todo |= (ab > 0.0 && g.x * g.x + g.y * g.y > I.tol2 * ab) ? 1 : 0;
          }
        }
        if (!__syncthreads_or(todo)) continue;
        if (tid == 0) P.flags[e * U1_MAXSWEEP + sweep] = 1;
        const int cur = evd_phase(Hs, Qs, Rm, sp, sq, I.nb > 0 ? U1_PB : U1_PB / 2, I.tol2);
        update_phase(stages, Qs + cur * (SV_W * SV_HLD), I);
      }
      base += (unsigned)npair + gridDim.x;
      grid.sync();
    }
    // ---- convergence: stop when no sector rotated in this sweep
    int any = 0;
    for (int bi = tid; bi < nblk; bi += U1_SVD_THREADS) any |= __ldcg(&P.flags[P.blk[bi] * U1_MAXSWEEP + sweep]);
    if (!__syncthreads_or(any)) { ++sweep; break; }
  }
  if (blockIdx.x == 0 && tid == 0) {
    atomicMax(&S.err[1], sweep);
    if (sweep >= U1_MAXSWEEP) {
      int bad = 0;
      for (int bi = 0; bi < nblk; ++bi) bad += P.flags[P.blk[bi] * U1_MAXSWEEP + U1_MAXSWEEP - 1];
      if (bad) atomicAdd(&S.err[2], bad);
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
  (void)G;
  DevState s = S; Plan p = P;
  void* args[] = {&s, &p};
  L.prof->begin(U1_ST_SVD, L.stream);
  cudaError_t err = cudaLaunchCooperativeKernel((void*)svd_kernel, dim3(L.svd_grid), dim3(U1_SVD_THREADS), args,
                                                (size_t)L.svd_smem, L.stream);
  L.prof->end(L.stream);
  if (err != cudaSuccess) return err;
  L.prof->begin(U1_ST_SORT, L.stream);
  sigma_sort_kernel<<<L.sms * 2, SORT_THREADS, U1MPS_SORT_MAX * 12, L.stream>>>(P);
  L.prof->end(L.stream);
  *L.launches += 2;
  return cudaGetLastError();
}
