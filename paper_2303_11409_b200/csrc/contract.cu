// contract.cu — step a2: the grouped complex128 block contraction of Eq.16:
//   Theta(c)[rows of c_l, cols of c_r] = lamL[c_l] * ( sum_{c'} U[(c_l-c, c-c_r),(c_l-c', c'-c_r)]
//                                         * Gamma^[s][c_l,c'] * lamC[c'] * Gamma^[s+1][c',c_r] ) * lamR[c_r]
// One persistent grid walks the tile list built by the planner (variable-size sectors of all
// gates of the chunk).  The U entry is a scalar per K-chunk (the delta functions of Eq.16 "tell us
// which entry of the unitary matrix to look up", L121), folded into the A operand together with
// lambda^[k]; lambda^[k-1], lambda^[k+1] are applied in the epilogue.  The result is written straight
// into the stacked column-major Jacobi matrix of the sector: Theta(c) if rows >= cols, else its
// conjugate transpose, with the identity (accumulator of the right singular vectors) below it.
#include "common.cuh"

#define KC 16
#define CT_THREADS 256

__device__ __forceinline__ cplx cmul(cplx a, cplx b) { return make_double2(a.x * b.x - a.y * b.y, a.x * b.y + a.y * b.x); }
__device__ __forceinline__ void cfma(cplx& acc, cplx a, cplx b) {
  acc.x = fma(a.x, b.x, acc.x); acc.x = fma(-a.y, b.y, acc.x);
  acc.y = fma(a.x, b.y, acc.y); acc.y = fma(a.y, b.x, acc.y);
}

// largest idx in [0, n) with pref[idx] <= v  (pref non-decreasing, pref[0] = 0 <= v < pref[n])
__device__ __forceinline__ int upper_entry(const int* __restrict__ pref, int n, int v) {
  int lo = 0, hi = n;  // invariant: pref[lo] <= v < pref[hi]
  while (hi - lo > 1) {
    int mid = (lo + hi) >> 1;
    if (pref[mid] <= v) lo = mid; else hi = mid;
  }
  return lo;
}

__global__ void __launch_bounds__(CT_THREADS) contract_kernel(DevState S, Plan P, int G) {
  __shared__ cplx As[KC][U1_TILE + 1];
  __shared__ cplx Bs[KC][U1_TILE];
  const int NC = S.NC, d = S.d, dd = d * d, N = S.N;
  const int nf = G * NC * dd;
  const int total = P.cnt[4];
  const int tid = threadIdx.x, tx = tid & 15, ty = tid >> 4;
  for (int tile = blockIdx.x; tile < total; tile += gridDim.x) {
    const int f = upper_entry(P.t2pref, nf, tile);
    const int e = f / dd, i = (f / d) % d, j = f % d;
    const int g = e / NC, c = e % NC, s = P.site[g];
    const int cl = c + i, cr = c - j;
    const int* nbL = S.nb + (long long)s * NC;
    const int* nbC = S.nb + (long long)(s + 1) * NC;
    const int* nbR = S.nb + (long long)(s + 2) * NC;
    const int nL = nbL[cl], nR = nbR[cr];
    const int tcols = u1_ceil_div(nR, U1_TILE);
    const int local = tile - P.t2pref[f];
    const int a0 = (local / tcols) * U1_TILE, b0 = (local % tcols) * U1_TILE;
    const cplx* Ug = P.U + (long long)g * dd * dd + (long long)(i * d + j) * dd;  // row (out_s = i, out_{s+1} = j)
    const cplx* gA = S.gam + (long long)s * S.gcap;
    const cplx* gB = S.gam + (long long)(s + 1) * S.gcap;
    cplx acc[2][2];
    acc[0][0] = acc[0][1] = acc[1][0] = acc[1][1] = make_double2(0.0, 0.0);
    const int cplo = max(max(cr, cl - d + 1), 0), cphi = min(min(cl, cr + d - 1), N);
    for (int cp = cplo; cp <= cphi; ++cp) {  // old centre sectors c' (the alpha_k sum of Eq.16, sector by sector)
      const int nC = nbC[cp];
      if (nC == 0) continue;
      const cplx u = Ug[(cl - cp) * d + (cp - cr)];
      const cplx* A = gA + S.gamoff[((long long)s * NC + cl) * d + (cl - cp)];       // nL x nC
      const cplx* B = gB + S.gamoff[((long long)(s + 1) * NC + cp) * d + (cp - cr)];  // nC x nR
      const double* lamC = S.lam + (long long)(s + 1) * S.chi + S.ob[(long long)(s + 1) * NC + cp];
      for (int k0 = 0; k0 < nC; k0 += KC) {
        __syncthreads();
        {  // A tile: k fastest
          const int k = tid & (KC - 1);
          for (int a = tid / KC; a < U1_TILE; a += CT_THREADS / KC) {
            cplx v = make_double2(0.0, 0.0);
            if (a0 + a < nL && k0 + k < nC) {
              v = A[(long long)(a0 + a) * nC + k0 + k];
              const double l = lamC[k0 + k];
              v = cmul(v, make_double2(u.x * l, u.y * l));
            }
            As[k][a] = v;
          }
          const int b = tid & (U1_TILE - 1);
          for (int kk = tid / U1_TILE; kk < KC; kk += CT_THREADS / U1_TILE) {
            cplx v = make_double2(0.0, 0.0);
            if (b0 + b < nR && k0 + kk < nC) v = B[(long long)(k0 + kk) * nR + b0 + b];
            Bs[kk][b] = v;
          }
        }
        __syncthreads();
#pragma unroll
        for (int k = 0; k < KC; ++k) {
          const cplx x0 = As[k][ty * 2], x1 = As[k][ty * 2 + 1];
          const cplx y0 = Bs[k][tx * 2], y1 = Bs[k][tx * 2 + 1];
          cfma(acc[0][0], x0, y0); cfma(acc[0][1], x0, y1);
          cfma(acc[1][0], x1, y0); cfma(acc[1][1], x1, y1);
        }
      }
    }
    // epilogue: lambda^[k-1] on rows, lambda^[k+1] on columns, write into the stacked Jacobi matrix
    int rowoff = 0, coloff = 0;
    for (int ii = 0; ii < i; ++ii) rowoff += nbL[c + ii];
    for (int jj = d - 1; jj > j; --jj) if (c - jj >= 0) coloff += nbR[c - jj];  // column blocks ascending c_r
    const double* lamL = S.lam + (long long)s * S.chi + S.ob[(long long)s * NC + cl];
    const double* lamR = S.lam + (long long)(s + 2) * S.chi + S.ob[(long long)(s + 2) * NC + cr];
    const int rows = P.rows[e], cols = P.cols[e];
    const bool tr = rows < cols;
    const int ld = rows + cols;  // m + n
    cplx* Wd = P.W + P.goff[e];
#pragma unroll
    for (int aa = 0; aa < 2; ++aa)
#pragma unroll
      for (int bb = 0; bb < 2; ++bb) {
        const int a = a0 + ty * 2 + aa, b = b0 + tx * 2 + bb;
        if (a < nL && b < nR) {
          const double sc = lamL[a] * lamR[b];
          cplx v = make_double2(acc[aa][bb].x * sc, acc[aa][bb].y * sc);
          const long long r = rowoff + a, q = coloff + b;
          if (!tr) Wd[r + q * ld] = v;
          else Wd[q + r * ld] = make_double2(v.x, -v.y);
        }
      }
  }
}

// Identity below every Theta block: rows m..m+n-1 of the stacked matrix (accumulates the rotations).
__global__ void identity_kernel(Plan P) {
  const int nblk = P.cnt[0];
  for (int bi = blockIdx.x; bi < nblk; bi += gridDim.x) {
    const int e = P.blk[bi];
    const int rows = P.rows[e], cols = P.cols[e];
    const int m = max(rows, cols), n = min(rows, cols), ld = m + n;
    cplx* Wd = P.W + P.goff[e];
    for (long long idx = threadIdx.x; idx < (long long)n * n; idx += blockDim.x) {
      const int r = (int)(idx % n), q = (int)(idx / n);
      Wd[(long long)q * ld + m + r] = make_double2(r == q ? 1.0 : 0.0, 0.0);
    }
  }
}

void u1_launch_contract(const DevState& S, const Plan& P, int G, const LaunchCfg& L) {
  L.prof->begin(U1_ST_CONTRACT, L.stream);
  contract_kernel<<<L.sms * 4, CT_THREADS, 0, L.stream>>>(S, P, G);
  L.prof->end(L.stream);
  L.prof->begin(U1_ST_IDENTITY, L.stream);
  identity_kernel<<<L.sms * 2, 256, 0, L.stream>>>(P);
  L.prof->end(L.stream);
  *L.launches += 2;
}
