// contract.cu — step a2: the grouped complex128 block contraction of Eq.16:
//   Theta(c)[rows of c_l, cols of c_r] = lamL[c_l] * ( sum_{c'} U[(c_l-c, c-c_r),(c_l-c', c'-c_r)]
//                                         * Gamma^[s][c_l,c'] * lamC[c'] * Gamma^[s+1][c',c_r] ) * lamR[c_r]
// One persistent grid walks the tile list built by the planner (variable-size sectors of all
// gates of the chunk), 32 x 32 output tiles on FP64 tensor tiles (DMMA.8x8x4, 4 real MMAs per complex product).
// Minimum form: T(c') = Gamma^[s][c_l,c'] lamC[c'] Gamma^[s+1][c',c_r] is formed once per block pair (c_l, c_r) and
// mixed into every Theta(c) with its U entry (the delta functions of Eq.16 "tell us which entry of the unitary matrix
// to look up", L121); lambda^[k] is folded into the A operand, lambda^[k-1], lambda^[k+1] are applied in the epilogue.  The result is written straight
// into the stacked column-major Jacobi matrix of the sector: Theta(c) if rows >= cols, else its
// conjugate transpose, with the identity (accumulator of the right singular vectors) below it.
#include "common.cuh"

#define KC 16          // K-chunk (columns of A / rows of B) per stage
#define CT_THREADS 128 // 4 warps: warp w owns rows 8w..8w+7 of the 32 x 32 output tile (4 DMMA tiles of 8 x 8)
#define CT_RUN 4       // consecutive tiles per work-queue step
#define CT_LD 34       // shared-memory leading dimension (complex elements), 2 mod 8: conflict-free LDS.128 fragments

__device__ __forceinline__ cplx cmul(cplx a, cplx b) { return make_double2(a.x * b.x - a.y * b.y, a.x * b.y + a.y * b.x); }

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
  __shared__ __align__(16) cplx As[KC * CT_LD];   // As[k][a]: lamC[k] A[a0 + a][k0 + k]
  __shared__ __align__(16) cplx Bs[KC * CT_LD];   // Bs[k][b]: B[k0 + k][b0 + b]
  const int NC = S.NC, d = S.d, dd = d * d, N = S.N;
  const int nf = G * NC * dd;
  const int total = P.cnt[4];
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5, lr = lane >> 2, lk = lane & 3;
  // tiles are handed out in runs of CT_RUN consecutive tiles: one binary search of the tile prefix per run, then a
  // linear advance
  for (int run = blockIdx.x; run * CT_RUN < total; run += gridDim.x) {
   int f = upper_entry(P.t2pref, nf, run * CT_RUN);
   for (int tile = run * CT_RUN; tile < min(total, (run + 1) * CT_RUN); ++tile) {
    while (P.t2pref[f + 1] <= tile) ++f;
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
    const cplx* Ug = P.U + (long long)g * dd * dd;
    const cplx* gA = S.gam + (long long)s * S.gcap;
    const cplx* gB = S.gam + (long long)(s + 1) * S.gcap;
    // Minimum form of Eq.16: the block pair (c_l, c_r) occurs in Theta(c) for every c in [cplo, cphi], and the old centre
    // charges c' run over the same range; T(c') = Gamma^[s][c_l,c'] lamC[c'] Gamma^[s+1][c',c_r] does not depend on c.
    // The tile of the LOWEST c owns the pair: it forms each T(c') once and adds U[(c_l-c, c-c_r),(c_l-c', c'-c_r)] T(c')
    // into the tile of every Theta(c) (first c' written, later ones read-modify-write by the same thread); the tiles of
    // the other c have nothing to do.
    const int cplo = max(max(cr, cl - d + 1), 0), cphi = min(min(cl, cr + d - 1), N);
    if (c != cplo) continue;   // uniform over the CTA
    const double* lamL = S.lam + (long long)s * S.chi + S.ob[(long long)s * NC + cl];
    const double* lamR = S.lam + (long long)(s + 2) * S.chi + S.ob[(long long)(s + 2) * NC + cr];
    bool first = true;
    for (int cp = cplo; cp <= cphi + 1; ++cp) {  // old centre sectors c' (the alpha_k sum of Eq.16, sector by sector)
      const bool flush = cp > cphi;              // after the last c': blocks that no c' reached are written as zeros
      const int nC = flush ? 0 : nbC[cp];
      if (flush ? !first : nC == 0) continue;
      double cre[4][2], cim[4][2];
#pragma unroll
      for (int u = 0; u < 4; ++u) { cre[u][0] = cre[u][1] = 0.0; cim[u][0] = cim[u][1] = 0.0; }
      if (!flush) {
      const cplx* A = gA + S.gamoff[((long long)s * NC + cl) * d + (cl - cp)];       // nL x nC
      const cplx* B = gB + S.gamoff[((long long)(s + 1) * NC + cp) * d + (cp - cr)];  // nC x nR
      const double* lamC = S.lam + (long long)(s + 1) * S.chi + S.ob[(long long)(s + 1) * NC + cp];
      for (int k0 = 0; k0 < nC; k0 += KC) {
        // global -> registers (A: k fastest, B: b fastest: both coalesced), scale A by lamC[k]
        cplx ra[4], rb[4];
        {
          const int k = tid & (KC - 1);
#pragma unroll
          for (int x = 0; x < 4; ++x) {
            const int a = (tid >> 4) + 8 * x;
            cplx v = make_double2(0.0, 0.0);
            if (a0 + a < nL && k0 + k < nC) {
              const double l = lamC[k0 + k];
              v = A[(long long)(a0 + a) * nC + k0 + k];
              v.x *= l; v.y *= l;
            }
            ra[x] = v;
          }
          const int b = tid & (U1_TILE - 1);
#pragma unroll
          for (int x = 0; x < 4; ++x) {
            const int kk = (tid >> 5) + 4 * x;
            cplx v = make_double2(0.0, 0.0);
            if (b0 + b < nR && k0 + kk < nC) v = B[(long long)(k0 + kk) * nR + b0 + b];
            rb[x] = v;
          }
        }
        __syncthreads();  // the previous chunk has been consumed
        {
          const int k = tid & (KC - 1), b = tid & (U1_TILE - 1);
#pragma unroll
          for (int x = 0; x < 4; ++x) {
            As[k * CT_LD + (tid >> 4) + 8 * x] = ra[x];
            Bs[((tid >> 5) + 4 * x) * CT_LD + b] = rb[x];
          }
        }
        __syncthreads();
        const int nk = (min(KC, nC - k0) + 3) >> 2;
        for (int ks = 0; ks < nk; ++ks) {
          const cplx av = As[(4 * ks + lk) * CT_LD + 8 * warp + lr];
          const double nai = -av.y;
#pragma unroll
          for (int t = 0; t < 4; ++t) {
            const cplx bv = Bs[(4 * ks + lk) * CT_LD + 8 * t + lr];
            // a * b : re = ar br - ai bi ; im = ar bi + ai br
            dmma(cre[t][0], cre[t][1], av.x, bv.x); dmma(cre[t][0], cre[t][1], nai, bv.y);
            dmma(cim[t][0], cim[t][1], av.x, bv.y); dmma(cim[t][0], cim[t][1], av.y, bv.x);
          }
        }
      }
      __syncthreads();  // before the next c' (or the next tile) refills the stages
      }   // (!flush)
      // mix T(c') into every Theta(cc): lambda^[k-1] on rows, lambda^[k+1] on columns, into the stacked Jacobi matrices
      for (int cc = cplo; cc <= cphi; ++cc) {
        const int ec = g * NC + cc, ic = cl - cc, jc = cc - cr;
        const cplx uu = flush ? make_double2(0.0, 0.0) : Ug[(long long)(ic * d + jc) * dd + (cl - cp) * d + (cp - cr)];
        int rowoff = 0, coloff = 0;
        for (int ii = 0; ii < ic; ++ii) rowoff += nbL[cc + ii];
        for (int jj = d - 1; jj > jc; --jj) if (cc - jj >= 0) coloff += nbR[cc - jj];  // column blocks ascending c_r
        const int rows = P.rows[ec], cols = P.cols[ec];
        const bool tr = rows < cols;
        const int ld = rows + cols;  // m + n
        cplx* Wd = P.W + P.goff[ec];
        const int a = a0 + 8 * warp + lr;
        if (a < nL) {
          const double la = lamL[a];
#pragma unroll
          for (int t = 0; t < 4; ++t)
#pragma unroll
            for (int x = 0; x < 2; ++x) {
              const int b = b0 + 8 * t + 2 * lk + x;
              if (b < nR) {
                const double sc = la * lamR[b];
                const double tr_ = cre[t][x] * sc, ti_ = cim[t][x] * sc;
                cplx v = make_double2(uu.x * tr_ - uu.y * ti_, uu.x * ti_ + uu.y * tr_);
                const long long r = rowoff + a, q = coloff + b;
                cplx* dst = !tr ? &Wd[r + q * ld] : &Wd[q + r * ld];
                if (tr) v.y = -v.y;
                if (!first) { const cplx o = *dst; v.x += o.x; v.y += o.y; }
                *dst = v;
              }
            }
        }
      }
      first = false;
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
  contract_kernel<<<L.sms * 8, CT_THREADS, 0, L.stream>>>(S, P, G);
  L.prof->end(L.stream);
  L.prof->begin(U1_ST_IDENTITY, L.stream);
  identity_kernel<<<L.sms * 2, 256, 0, L.stream>>>(P);
  L.prof->end(L.stream);
  *L.launches += 2;
}
