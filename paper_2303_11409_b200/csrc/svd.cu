// svd.cu — step a3: one SVD per centre-charge sector ("Singular value decompositions are
// then performed on each Theta(c^[k])"; Eq.12), for all sectors of all gates of the chunk at once.
// The paper calls a library SVD (L131); here it is a batched one-sided (Hestenes) Jacobi SVD:
// the columns of the stacked matrix [G; J] (G = Theta(c) or its conjugate transpose so that
// m >= n, J = identity) are rotated pairwise until the columns of G are mutually orthogonal; then
// sigma_j = |G_j|, left vectors G_j / sigma_j, right vectors J_j.
// Blocking: columns are grouped in panels of b <= 16; a work item is a panel pair, staged in shared
// memory when it fits (else rotated in place through L2), one warp per column pair, warp-shuffle
// reductions for the three inner products of a rotation.  A persistent cooperative grid walks
// the round-robin tournament of panel pairs of every sector in lock step (one grid sync per round);
// convergence is decided on the device per sector, no host round trip.
#include <cooperative_groups.h>
#include "common.cuh"
namespace cg = cooperative_groups;

__device__ __forceinline__ double warp_sum(double v) {
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
  return v;
}

template <bool GLOBAL>
__device__ __forceinline__ cplx ldc(const cplx* p) {
  if (GLOBAL) return __ldcg(p);
  return *p;
}

// One Jacobi rotation of columns x, y (x has the lower column index) by one warp.
// Inner products over the top m rows (G part); the rotation is applied to all mt = m + n rows.
// Returns true if a rotation was applied.
template <bool GLOBAL>
__device__ __forceinline__ bool rotate_pair(cplx* x, cplx* y, int m, int mt, int lane, double tol2) {
  double a = 0.0, b = 0.0, gr = 0.0, gi = 0.0;
  for (int r = lane; r < m; r += 32) {
    const cplx xv = ldc<GLOBAL>(x + r), yv = ldc<GLOBAL>(y + r);
    a = fma(xv.x, xv.x, a); a = fma(xv.y, xv.y, a);
    b = fma(yv.x, yv.x, b); b = fma(yv.y, yv.y, b);
    gr = fma(xv.x, yv.x, gr); gr = fma(xv.y, yv.y, gr);   // gamma = x^H y
    gi = fma(xv.x, yv.y, gi); gi = fma(-xv.y, yv.x, gi);
  }
  a = warp_sum(a); b = warp_sum(b); gr = warp_sum(gr); gi = warp_sum(gi);
  const double g2 = gr * gr + gi * gi;
  const double hi = fmax(a, b), lo = fmin(a, b);
  if (!(lo > 0.0) || lo < 1e-40 * hi || g2 <= tol2 * a * b) return false;
  const double ag = sqrt(g2);
  const double zeta = (b - a) / (2.0 * ag);
  const double t = copysign(1.0, zeta) / (fabs(zeta) + sqrt(1.0 + zeta * zeta));
  const double cs = rsqrt(1.0 + t * t);
  const double sn = cs * t;
  const double sr = sn * gr / ag, si = sn * gi / ag;  // s = sn * e^{i phi}
  const bool swp = (a - t * ag) < (b + t * ag);       // keep the larger norm in the lower column
  for (int r = lane; r < mt; r += 32) {
    const cplx xv = ldc<GLOBAL>(x + r), yv = ldc<GLOBAL>(y + r);
    // x' = cs x - conj(s) y ;  y' = s x + cs y
    cplx xn, yn;
    xn.x = cs * xv.x - (sr * yv.x + si * yv.y);
    xn.y = cs * xv.y - (sr * yv.y - si * yv.x);
    yn.x = cs * yv.x + (sr * xv.x - si * xv.y);
    yn.y = cs * yv.y + (sr * xv.y + si * xv.x);
    if (swp) { x[r] = yn; y[r] = xn; } else { x[r] = xn; y[r] = yn; }
  }
  return true;
}

struct BlkInfo { int m, n, mt, b, in_smem, np; cplx* W; double tol2; };

__device__ __forceinline__ BlkInfo blk_info(const Plan& P, int e, long long smem_elems) {
  BlkInfo B;
  const int r = P.rows[e], q = P.cols[e];
  B.m = max(r, q); B.n = min(r, q); B.mt = B.m + B.n;
  B.b = u1_panel_width(B.mt, B.n, smem_elems, &B.in_smem);
  B.np = u1_ceil_div(B.n, B.b);
  B.W = P.W + P.goff[e];
  const double tol = sqrt((double)B.m) * 2.3e-16;
  B.tol2 = tol * tol;
  return B;
}

// circle-method round robin over np2 (even) players: slot k of round t -> (a, b)
__device__ __forceinline__ void rr_pair(int t, int k, int np2, int* a, int* b) {
  const int q = np2 - 1;
  if (k == 0) { *a = t % q; *b = q; }
  else { *a = (t + k) % q; *b = (t - k + 2 * q) % q; }
  if (*a > *b) { int s = *a; *a = *b; *b = s; }
}

__global__ void __launch_bounds__(U1_SVD_THREADS, 1) svd_kernel(DevState S, Plan P, int G, long long smem_elems) {
  extern __shared__ __align__(16) unsigned char smraw[];
  cplx* sm = reinterpret_cast<cplx*>(smraw);
  __shared__ int s_rot;
  cg::grid_group grid = cg::this_grid();
  const int nblk = P.cnt[0], npair = P.cnt[1], nintra = P.cnt[2], maxP = P.cnt[3];
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  int sweep = 0;
  for (; sweep < U1_MAXSWEEP; ++sweep) {
    // ---- intra-panel phase: all pairs inside one panel
    for (int it = blockIdx.x; it < nintra; it += gridDim.x) {
      const int e = P.iitem_e[it], p = P.iitem_p[it];
      if (sweep > 0 && __ldcg(&P.flags[e * U1_MAXSWEEP + sweep - 1]) == 0) continue;  // sector converged
      const BlkInfo B = blk_info(P, e, smem_elems);
      const int c0 = p * B.b, nc = min(B.b, B.n - c0);
      if (nc < 2) continue;
      const int nce = nc + (nc & 1);
      __syncthreads();
      if (tid == 0) s_rot = 0;
      if (B.in_smem) {
        for (long long idx = tid; idx < (long long)nc * B.mt; idx += U1_SVD_THREADS)
          sm[idx] = __ldcg(B.W + (long long)c0 * B.mt + idx);
      }
      __syncthreads();
      bool rot = false;
      for (int st = 0; st < nce - 1; ++st) {
        if (warp < nce / 2) {
          int a, b;
          rr_pair(st, warp, nce, &a, &b);
          if (b < nc) {
            if (B.in_smem) rot |= rotate_pair<false>(sm + (long long)a * B.mt, sm + (long long)b * B.mt, B.m, B.mt, lane, B.tol2);
            else rot |= rotate_pair<true>(B.W + (long long)(c0 + a) * B.mt, B.W + (long long)(c0 + b) * B.mt, B.m, B.mt, lane, B.tol2);
          }
        }
        __syncthreads();
      }
      if (rot && lane == 0) s_rot = 1;
      __syncthreads();
      if (s_rot) {
        if (B.in_smem)
          for (long long idx = tid; idx < (long long)nc * B.mt; idx += U1_SVD_THREADS)
            B.W[(long long)c0 * B.mt + idx] = sm[idx];
        if (tid == 0) P.flags[e * U1_MAXSWEEP + sweep] = 1;
      }
    }
    grid.sync();
    // ---- panel-pair rounds
    for (int t = 0; t < maxP - 1; ++t) {
      for (int it = blockIdx.x; it < npair; it += gridDim.x) {
        const int e = P.pitem_e[it], k = P.pitem_k[it];
        if (sweep > 0 && __ldcg(&P.flags[e * U1_MAXSWEEP + sweep - 1]) == 0) continue;
        const BlkInfo B = blk_info(P, e, smem_elems);
        const int np2 = B.np + (B.np & 1);
        if (t >= np2 - 1) continue;
        int pa, pb;
        rr_pair(t, k, np2, &pa, &pb);
        if (pb >= B.np) continue;  // bye
        const int ca = pa * B.b, cb = pb * B.b;
        const int na = min(B.b, B.n - ca), nbq = min(B.b, B.n - cb);
        __syncthreads();
        if (tid == 0) s_rot = 0;
        cplx* smB = sm + (long long)B.b * B.mt;
        if (B.in_smem) {
          for (long long idx = tid; idx < (long long)na * B.mt; idx += U1_SVD_THREADS)
            sm[idx] = __ldcg(B.W + (long long)ca * B.mt + idx);
          for (long long idx = tid; idx < (long long)nbq * B.mt; idx += U1_SVD_THREADS)
            smB[idx] = __ldcg(B.W + (long long)cb * B.mt + idx);
        }
        __syncthreads();
        bool rot = false;
        for (int st = 0; st < B.b; ++st) {
          if (warp < B.b) {
            const int i = warp, j = (warp + st) % B.b;
            if (i < na && j < nbq) {
              if (B.in_smem) rot |= rotate_pair<false>(sm + (long long)i * B.mt, smB + (long long)j * B.mt, B.m, B.mt, lane, B.tol2);
              else rot |= rotate_pair<true>(B.W + (long long)(ca + i) * B.mt, B.W + (long long)(cb + j) * B.mt, B.m, B.mt, lane, B.tol2);
            }
          }
          __syncthreads();
        }
        if (rot && lane == 0) s_rot = 1;
        __syncthreads();
        if (s_rot) {
          if (B.in_smem) {
            for (long long idx = tid; idx < (long long)na * B.mt; idx += U1_SVD_THREADS)
              B.W[(long long)ca * B.mt + idx] = sm[idx];
            for (long long idx = tid; idx < (long long)nbq * B.mt; idx += U1_SVD_THREADS)
              B.W[(long long)cb * B.mt + idx] = smB[idx];
          }
          if (tid == 0) P.flags[e * U1_MAXSWEEP + sweep] = 1;
        }
      }
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
  int dev = 0, maxsm = 0;
  cudaError_t err = cudaGetDevice(&dev);
  if (err != cudaSuccess) return err;
  err = cudaDeviceGetAttribute(&maxsm, cudaDevAttrMaxSharedMemoryPerBlockOptin, dev);
  if (err != cudaSuccess) return err;
  int smem = maxsm - 2048;  // leave room for static shared memory
  smem -= smem % 16;
  err = cudaFuncSetAttribute(svd_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, smem);
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
  long long smem_elems = (long long)L.svd_smem / (long long)sizeof(cplx);
  DevState s = S; Plan p = P; int g = G;
  void* args[] = {&s, &p, &g, &smem_elems};
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
