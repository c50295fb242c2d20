// select.cu — steps a4 and a5.
// a4 ("the largest chi singular values out of all the singular values for all
// Theta(c^[k])'s and their corresponding bonds are retained"): pool (sigma, c, j) of one gate, drop
// sigma <= cutoff (reading S7), order by (sigma desc, c asc, j asc) (S8), keep the first chi (at
// least one).  Every sector is already sorted, so the global rank of an element is its own
// position plus, for every other sector, the number of elements that precede it (binary search).
// Then renormalise (S9), write the new sector table of the centre bond, lambda, the block offsets
// of the two sites.
// a5 (Eq.13/14, L94-104, reading S4): Gamma~[s][c_l,c] = V(c)[rows of c_l, :keep(c)] / lambda^[k-1],
// Gamma~[s+1][c,c_r] = W(c)[:keep(c), cols of c_r] / lambda^[k+1]; tiled transposing scatter.
#include "common.cuh"

#define SEL_THREADS 1024

// number of leading elements of the descending array a[0..n) that are > v (strict) or >= v
__device__ __forceinline__ int count_before(const double* __restrict__ a, int n, double v, bool inclusive) {
  int lo = 0, hi = n;  // first index where the predicate fails
  while (lo < hi) {
    const int mid = (lo + hi) >> 1;
    const double x = a[mid];
    if (inclusive ? (x >= v) : (x > v)) lo = mid + 1; else hi = mid;
  }
  return lo;
}

__global__ void __launch_bounds__(SEL_THREADS) select_kernel(DevState S, Plan P, int G, int chi, double cutoff, int* done_counter,
                                                              double* gate_w) {
  extern __shared__ int keep_sh[];  // [NC]
  __shared__ double red[2][SEL_THREADS / 32];
  __shared__ double s_w[2];
  __shared__ int s_top;
  __shared__ int s_last;
  if (S.err[0] != 0) return;   // the plan did not fit (U1_ERR_WORKSPACE): its offsets must not be used
  const int NC = S.NC, d = S.d, g = blockIdx.x, s = P.site[g], C = s + 1;
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  const int* svo = P.svoff + g * NC;
  const int base = svo[0], end = svo[NC];
  for (int c = tid; c < NC; c += SEL_THREADS) keep_sh[c] = 0;
  if (tid == 0) s_top = -1;
  __syncthreads();
  double wall = 0.0, wkept = 0.0;
  for (int p = base + tid; p < end; p += SEL_THREADS) {
    int lo = 0, hi = NC;  // sector of pooled element p
    while (hi - lo > 1) { const int mid = (lo + hi) >> 1; if (svo[mid] <= p) lo = mid; else hi = mid; }
    const int c = lo, j = p - svo[c];
    const double v = P.svs[p];
    int rank = j;
    for (int c2 = 0; c2 < NC; ++c2) {
      const int n2 = svo[c2 + 1] - svo[c2];
      if (n2 == 0 || c2 == c) continue;
      rank += count_before(P.svs + svo[c2], n2, v, c2 < c);
    }
    wall = fma(v, v, wall);
    if (rank == 0) s_top = c;
    if (v > cutoff && rank < chi) { wkept = fma(v, v, wkept); atomicMax(&keep_sh[c], j + 1); }
  }
  // deterministic block reduction of the two weights
  for (int o = 16; o > 0; o >>= 1) { wall += __shfl_xor_sync(0xffffffffu, wall, o); wkept += __shfl_xor_sync(0xffffffffu, wkept, o); }
  if (lane == 0) { red[0][warp] = wall; red[1][warp] = wkept; }
  __syncthreads();
  if (tid == 0) {
    double a = 0.0, b = 0.0;
    for (int w = 0; w < SEL_THREADS / 32; ++w) { a += red[0][w]; b += red[1][w]; }
    bool none = true;
    for (int c = 0; c < NC; ++c) none = none && keep_sh[c] == 0;
    if (none && s_top >= 0) {  // keep at least one: the globally largest (sigma, smallest c)
      keep_sh[s_top] = 1;
      const double v = P.svs[svo[s_top]];
      b = v * v;
    }
    s_w[0] = a; s_w[1] = b;
    gate_w[2 * g] = b; gate_w[2 * g + 1] = a;
    // new sector table of the centre bond
    int run = 0;
    for (int c = 0; c < NC; ++c) { S.nb[(long long)C * NC + c] = keep_sh[c]; S.ob[(long long)C * NC + c] = run; run += keep_sh[c]; P.keep[g * NC + c] = keep_sh[c]; }
    // block offsets of site s: blocks (cl, i), n_L(cl) x keep(cl - i)
    long long off = 0;
    const int* nbL = S.nb + (long long)s * NC;
    for (int cl = 0; cl < NC; ++cl)
      for (int i = 0; i < d; ++i) {
        S.gamoff[((long long)s * NC + cl) * d + i] = off;
        if (cl - i >= 0) off += (long long)nbL[cl] * keep_sh[cl - i];
      }
  }
  __syncthreads();
  if (tid == 0) {
    // block offsets of site s+1: blocks (c, j), keep(c) x n_R(c - j)
    long long off = 0;
    const int* nbR = S.nb + (long long)(s + 2) * NC;
    for (int c = 0; c < NC; ++c)
      for (int j = 0; j < d; ++j) {
        S.gamoff[((long long)(s + 1) * NC + c) * d + j] = off;
        if (c - j >= 0) off += (long long)keep_sh[c] * nbR[c - j];
      }
  }
  // lambda~ = sigma_kept / sqrt(w)
  const double isq = 1.0 / sqrt(s_w[1]);
  for (int p = base + tid; p < end; p += SEL_THREADS) {
    int lo = 0, hi = NC;
    while (hi - lo > 1) { const int mid = (lo + hi) >> 1; if (svo[mid] <= p) lo = mid; else hi = mid; }
    const int c = lo, j = p - svo[c];
    if (j < keep_sh[c]) {
      int o = 0;
      for (int c2 = 0; c2 < c; ++c2) o += keep_sh[c2];
      S.lam[(long long)C * S.chi + o + j] = P.svs[p] * isq;
    }
  }
  // the last CTA to finish adds the per-gate weights to the log-norm in gate order (deterministic)
  __threadfence();
  __syncthreads();
  if (tid == 0) s_last = (atomicAdd(done_counter, 1) == G - 1);
  __syncthreads();
  if (s_last && tid == 0) {
    __threadfence();
    double ln = S.scal[0], disc = S.scal[1];
    for (int gg = 0; gg < G; ++gg) {
      const double wk = __ldcg(&gate_w[2 * gg]), wa = __ldcg(&gate_w[2 * gg + 1]);
      ln += 0.5 * log(wk);
      disc += wa - wk;
      S.scal[2] = wk; S.scal[3] = wa;
    }
    S.scal[0] = ln; S.scal[1] = disc;
    *done_counter = 0;
  }
}

// a5 work list over (entry, part) restricted to sectors that KEEP singular vectors (the planner sized it before a4 had
// decided): strips of U1_TILE bond indices - rows of V(c), columns of W(c) - each strip runs over all kept vectors.
// One CTA, exclusive scan into P.t5pref.
__global__ void __launch_bounds__(SEL_THREADS) retile_kernel(Plan P, int L /* = 2 G NC */) {
  __shared__ int sh[SEL_THREADS];
  auto tiles = [&](int f) {
    const int e = f >> 1, k = P.keep[e];
    if (k == 0) return 0;
    return (f & 1) ? u1_ceil_div(P.cols[e], U1_TILE) : u1_ceil_div(P.rows[e], U1_TILE);
  };
  u1_block_excl_scan<int, SEL_THREADS>(tiles, P.t5pref, L, sh);
  if (threadIdx.x == 0) P.cnt[5] = P.t5pref[L];
}

#define SC_THREADS 256
#define SC_VW 64   // singular vectors per pass of a strip
// a5: V(c) (part 0) and W(c) (part 1) out of the stacked Jacobi matrices into the block-sparse Gammas, in strips of 32
// bond indices (rows a of V, columns b of W) x all kept singular vectors.  What is constant along a bond index -
// destination block, offset and 1/lambda (Eq.13/14) - is worked out once per strip by 32 threads; per pass of 64
// vectors another 64 threads fetch the source column and 1/sigma of each; the bulk is then load - multiply - store:
// coalesced 512-byte column segments in, 512- / 1024-byte row segments out (V is transposed through shared memory).
__global__ void __launch_bounds__(SC_THREADS) scatter_kernel(DevState S, Plan P, int G) {
  __shared__ cplx tile[SC_VW][U1_TILE + 1];
  __shared__ long long s_src[SC_VW];     // per singular vector jj: offset of its column in the stacked matrix (-1: not kept)
  __shared__ double s_isg[SC_VW];        // ... 1/sigma (or 1 where the vectors are the unit-norm J columns)
  __shared__ long long s_dst[U1_TILE];   // per bond index (row a of V / column b of W): destination offset (-1: outside)
  __shared__ double s_ilm[U1_TILE];      // ... 1/lambda of that bond index (Eq.13/14)
  __shared__ int s_ldd[U1_TILE];         // ... row length of the destination block (part 1)
  const int NC = S.NC, d = S.d;
  const int nf = G * NC * 2, total = P.cnt[5];
  const int tid = threadIdx.x, tx = tid & 31, ty = tid >> 5;
  for (int unit = blockIdx.x; unit < total; unit += gridDim.x) {
    int f;
    {
      int lo = 0, hi = nf;
      while (hi - lo > 1) { const int mid = (lo + hi) >> 1; if (P.t5pref[mid] <= unit) lo = mid; else hi = mid; }
      f = lo;
    }
    const int e = f >> 1, part = f & 1;
    const int g = e / NC, c = e % NC, s = P.site[g];
    const int rows = P.rows[e], cols = P.cols[e], m = max(rows, cols), n = min(rows, cols), ld = m + n;
    const bool tr = rows < cols;
    const int keep = P.keep[e];
    const cplx* W = P.W + P.goff[e];
    const int so = P.svoff[e];
    const int i0 = (unit - P.t5pref[f]) * U1_TILE;   // first bond index of the strip
    __syncthreads();   // the previous strip is done with the shared arrays
    if (tid < U1_TILE) {  // bond index i0 + tid: row a of V (left bond) or column b of W (right bond)
      const int idx = i0 + tid;
      long long dst = -1; double ilm = 0.0; int ldd = 0;
      if (part == 0 && idx < rows) {
        const int* nbL = S.nb + (long long)s * NC;
        int i = 0, al = idx;
        while (al >= nbL[c + i]) { al -= nbL[c + i]; ++i; }
        const int cl = c + i;
        ilm = 1.0 / S.lam[(long long)s * S.chi + S.ob[(long long)s * NC + cl] + al];
        dst = (long long)s * S.gcap + S.gamoff[((long long)s * NC + cl) * d + i] + (long long)al * keep;
        ldd = keep;
      } else if (part == 1 && idx < cols) {
        const int* nbR = S.nb + (long long)(s + 2) * NC;
        int jq = d - 1, bl = idx;
        while (c - jq < 0) --jq;
        while (bl >= nbR[c - jq]) { bl -= nbR[c - jq]; --jq; }
        const int cr = c - jq;
        ilm = 1.0 / S.lam[(long long)(s + 2) * S.chi + S.ob[(long long)(s + 2) * NC + cr] + bl];
        dst = (long long)(s + 1) * S.gcap + S.gamoff[((long long)(s + 1) * NC + c) * d + (c - cr)] + bl;
        ldd = nbR[cr];
      }
      s_dst[tid] = dst; s_ilm[tid] = ilm; s_ldd[tid] = ldd;
    }
    for (int j0 = 0; j0 < keep; j0 += SC_VW) {
      __syncthreads();   // the previous pass is done with tile / s_src (and the strip's arrays are in place)
      if (tid >= SC_THREADS - SC_VW) {  // singular vector j0 + k
        const int k = tid - (SC_THREADS - SC_VW), pj = j0 + k;
        long long src = -1; double isg = 1.0;
        if (pj < keep) {
          src = (long long)P.perm[so + pj] * ld;
          // V = G / sigma when G holds Theta (rows >= cols), W = conj(G) / sigma when it holds Theta^H
          if ((part == 0) != tr) isg = 1.0 / P.svs[so + pj];
        }
        s_src[k] = src; s_isg[k] = isg;
      }
      __syncthreads();
      if (part == 0) {
        // V(c)[a, jj] = G[a, p] / sigma (rows >= cols) or J[a, p]: read 32 rows of 64 columns, transpose, write rows
        const int roff = tr ? m : 0;
        cplx v[SC_VW / (SC_THREADS / 32)];   // all loads of the pass in flight before the first use
#pragma unroll
        for (int x = 0; x < SC_VW / (SC_THREADS / 32); ++x) {
          const long long src = s_src[ty + x * (SC_THREADS / 32)];
          v[x] = (src >= 0 && i0 + tx < rows) ? __ldcs(W + src + roff + i0 + tx) : make_double2(0.0, 0.0);
        }
#pragma unroll
        for (int x = 0; x < SC_VW / (SC_THREADS / 32); ++x) {
          const int jj = ty + x * (SC_THREADS / 32);
          const double sc = s_isg[jj];
          tile[jj][tx] = make_double2(v[x].x * sc, v[x].y * sc);
        }
        __syncthreads();
        for (int aa = ty; aa < U1_TILE; aa += SC_THREADS / 32) {
          const long long dst = s_dst[aa];
          const double il = s_ilm[aa];
#pragma unroll
          for (int h = 0; h < SC_VW / 32; ++h) {
            const int jj = tx + 32 * h;
            if (dst >= 0 && j0 + jj < keep) {
              cplx v = tile[jj][aa];
              v.x *= il; v.y *= il;
              __stcs(&S.gam[dst + j0 + jj], v);
            }
          }
        }
      } else {
        // W(c)[jj, b] = conj(J[b, p]) (rows >= cols) or conj(G[b, p]) / sigma: no transposition needed
        const int roff = tr ? 0 : m;
        const long long dst = s_dst[tx];
        const double il = s_ilm[tx];
        const int ldd = s_ldd[tx];
        cplx v[SC_VW / (SC_THREADS / 32)];
#pragma unroll
        for (int x = 0; x < SC_VW / (SC_THREADS / 32); ++x) {
          const long long src = s_src[ty + x * (SC_THREADS / 32)];
          v[x] = (src >= 0 && dst >= 0) ? __ldcs(W + src + roff + i0 + tx) : make_double2(0.0, 0.0);
        }
#pragma unroll
        for (int x = 0; x < SC_VW / (SC_THREADS / 32); ++x) {
          const int jj = ty + x * (SC_THREADS / 32);
          if (s_src[jj] >= 0 && dst >= 0) {
            const double sc = s_isg[jj] * il;
            __stcs(&S.gam[dst + (long long)(j0 + jj) * ldd], make_double2(v[x].x * sc, -v[x].y * sc));
          }
        }
      }
    }
  }
}

void u1_launch_select_scatter(const DevState& S, const Plan& P, int G, int chi, double cutoff, const LaunchCfg& L) {
  int* counter = P.cnt + 7;
  L.prof->begin(U1_ST_SELECT, L.stream);
  select_kernel<<<G, SEL_THREADS, S.NC * sizeof(int), L.stream>>>(S, P, G, chi, cutoff, counter, P.gate_w);
  L.prof->end(L.stream);
  L.prof->begin(U1_ST_SCATTER, L.stream);
  retile_kernel<<<1, SEL_THREADS, 0, L.stream>>>(P, 2 * G * S.NC);
  scatter_kernel<<<L.sms * 8, SC_THREADS, 0, L.stream>>>(S, P, G);
  L.prof->end(L.stream);
  *L.launches += 3;
}
