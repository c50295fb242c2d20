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

#define SC_THREADS 256
__global__ void __launch_bounds__(SC_THREADS) scatter_kernel(DevState S, Plan P, int G) {
  __shared__ cplx tile[U1_TILE][U1_TILE + 1];
  const int NC = S.NC, d = S.d;
  const int nf = G * NC * 2, total = P.cnt[5];
  const int tid = threadIdx.x, tx = tid & 31, ty = tid >> 5;
  for (int t = blockIdx.x; t < total; t += gridDim.x) {
    int lo = 0, hi = nf;
    while (hi - lo > 1) { const int mid = (lo + hi) >> 1; if (P.t5pref[mid] <= t) lo = mid; else hi = mid; }
    const int f = lo, e = f >> 1, part = f & 1;
    const int g = e / NC, c = e % NC, s = P.site[g];
    const int rows = P.rows[e], cols = P.cols[e], m = max(rows, cols), n = min(rows, cols), ld = m + n;
    const bool tr = rows < cols;
    const int keep = P.keep[e];
    const int local = t - P.t5pref[f];
    const cplx* W = P.W + P.goff[e];
    const int so = P.svoff[e];
    if (part == 0) {
      // V(c)[a, jj]: case A (rows >= cols) = G[a, p] / sigma_p ; case B = J[a, p]
      const int tcols = u1_ceil_div(n, U1_TILE);
      const int a0 = (local / tcols) * U1_TILE, j0 = (local % tcols) * U1_TILE;
      if (j0 >= keep) continue;
      __syncthreads();
      for (int jj = ty; jj < U1_TILE; jj += SC_THREADS / 32) {
        const int pj = j0 + jj, a = a0 + tx;
        cplx v = make_double2(0.0, 0.0);
        if (pj < keep && a < rows) {
          const int p = P.perm[so + pj];
          if (!tr) { const double is = 1.0 / P.svs[so + pj]; v = __ldcg(W + (long long)p * ld + a); v.x *= is; v.y *= is; }
          else v = __ldcg(W + (long long)p * ld + m + a);
        }
        tile[jj][tx] = v;
      }
      __syncthreads();
      const int* nbL = S.nb + (long long)s * NC;
      for (int aa = ty; aa < U1_TILE; aa += SC_THREADS / 32) {
        const int a = a0 + aa, pj = j0 + tx;
        if (a < rows && pj < keep) {
          int i = 0, al = a;
          while (al >= nbL[c + i]) { al -= nbL[c + i]; ++i; }
          const int cl = c + i;
          const double il = 1.0 / S.lam[(long long)s * S.chi + S.ob[(long long)s * NC + cl] + al];
          cplx v = tile[tx][aa];
          v.x *= il; v.y *= il;
          S.gam[(long long)s * S.gcap + S.gamoff[((long long)s * NC + cl) * d + i] + (long long)al * keep + pj] = v;
        }
      }
    } else {
      // W(c)[jj, b]: case A = conj(J[b, p]) ; case B = conj(G[b, p]) / sigma_p
      const int tcols = u1_ceil_div(cols, U1_TILE);
      const int j0 = (local / tcols) * U1_TILE, b0 = (local % tcols) * U1_TILE;
      if (j0 >= keep) continue;
      const int* nbR = S.nb + (long long)(s + 2) * NC;
      const int b = b0 + tx;
      int cr = 0, bl = b;
      if (b < cols) {
        int jq = d - 1;
        while (c - jq < 0) --jq;
        while (bl >= nbR[c - jq]) { bl -= nbR[c - jq]; --jq; }
        cr = c - jq;
      }
      for (int jj = ty; jj < U1_TILE; jj += SC_THREADS / 32) {
        const int pj = j0 + jj;
        if (pj < keep && b < cols) {
          const int p = P.perm[so + pj];
          cplx v;
          if (!tr) v = __ldcg(W + (long long)p * ld + m + b);
          else { const double is = 1.0 / P.svs[so + pj]; v = __ldcg(W + (long long)p * ld + b); v.x *= is; v.y *= is; }
          const double il = 1.0 / S.lam[(long long)(s + 2) * S.chi + S.ob[(long long)(s + 2) * NC + cr] + bl];
          v.x *= il; v.y *= -il;
          S.gam[(long long)(s + 1) * S.gcap + S.gamoff[((long long)(s + 1) * NC + c) * d + (c - cr)] + (long long)pj * nbR[cr] + bl] = v;
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
  scatter_kernel<<<L.sms * 4, SC_THREADS, 0, L.stream>>>(S, P, G);
  L.prof->end(L.stream);
  *L.launches += 2;
}
