// envs.cu — full-environment expectation values <psi|n_k|psi> / <psi|psi> of the U(1) MPS (SURVEY section 8(f)-4,
// PAPER.md Eq.15 L112-114 for the state, Eq.10 L74-80 for what "canonical" would mean): once truncation has broken the
// canonical form, the lambda-weighted formula of step a6 is only approximate, while the contraction with explicit left
// and right environments is exact for whatever Gamma, lambda the state holds.
//   A^[s](cl, cr) = Gamma^[s][cl, cr] diag(lambda^[s+1][cr])
//   E_0 = {N: [[1]]},  E_{s+1}[cr] = sum_cl A^H E_s[cl] A          (left environments, n x n per sector)
//   R_M = {0: [[1]]},  R_s[cl]     = sum_cr A R_{s+1}[cr] A^H      (right environments)
//   <n_s> = sum_{cl,cr} (cl - cr) tr(A^H E_s[cl] A R_{s+1}[cr]) / E_M[0]
// Everything is a grouped complex128 GEMM over the charge blocks of one site (FP64 DMMA tiles, as in step a2); the
// trace is an element-wise inner product of T = E_s Gamma and S = Gamma lambda R lambda.  The host knows the sector
// tables (the call synchronises anyway), builds the block descriptors of all stages once and uploads them; the device
// does all arithmetic.
#include <algorithm>
#include <vector>
#include "common.cuh"

#define EV_THREADS 128
#define EV_KC 16
#define EV_LD 34
#define EV_MAXTERM 8   // = U1MPS_D_MAX: a block sum runs over at most d occupations

struct EnvDesc {
  const cplx* A[EV_MAXTERM];     // term t: left operand, dense row-major (m x k, or k x m if opA)
  const cplx* B[EV_MAXTERM];     // ... right operand (k x n, or n x k if opB)
  const double* ks[EV_MAXTERM];  // ... optional scale over the inner index (nullptr: none)
  int k[EV_MAXTERM];
  double w[EV_MAXTERM];          // ... weight of the term (the occupation, for an inserted n)
  cplx* C;                       // m x n row-major
  const double* rs;              // optional output row / column scales
  const double* cs;
  double alpha;
  int m, n, nterm, opA, opB;     // op = 1: the operand is the conjugate transpose of what is stored
};

// C = alpha diag(rs) (sum_t op(A_t) diag(ks_t) op(B_t)) diag(cs), 32 x 32 output tiles, K-chunks of 16 through shared
// memory, 4 warps x one 8-row strip each, DMMA.8x8x4 (4 real products per complex one).
__global__ void __launch_bounds__(EV_THREADS) env_gemm_kernel(const EnvDesc* __restrict__ desc, const int* __restrict__ tpref, int ndesc) {
  __shared__ __align__(16) cplx As[EV_KC * EV_LD];   // As[kk][a]
  __shared__ __align__(16) cplx Bs[EV_KC * EV_LD];   // Bs[kk][b]
  const int total = tpref[ndesc];
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5, lr = lane >> 2, lk = lane & 3;
  for (int tile = blockIdx.x; tile < total; tile += gridDim.x) {
    int lo = 0, hi = ndesc;
    while (hi - lo > 1) { const int mid = (lo + hi) >> 1; if (tpref[mid] <= tile) lo = mid; else hi = mid; }
    const EnvDesc& D = desc[lo];
    const int m = D.m, n = D.n, tcols = u1_ceil_div(n, U1_TILE), local = tile - tpref[lo];
    const int a0 = (local / tcols) * U1_TILE, b0 = (local % tcols) * U1_TILE;
    double cre[4][2], cim[4][2];
#pragma unroll
    for (int u = 0; u < 4; ++u) { cre[u][0] = cre[u][1] = 0.0; cim[u][0] = cim[u][1] = 0.0; }
    for (int t = 0; t < D.nterm; ++t) {
      const cplx* A = D.A[t];
      const cplx* B = D.B[t];
      const double* ks = D.ks[t];
      const int K = D.k[t];
      const double wt = D.w[t];
      for (int k0 = 0; k0 < K; k0 += EV_KC) {
        cplx ra[4], rb[4];
        // A chunk: 32 (a) x 16 (kk)
        if (!D.opA) {   // stored m x K: kk fastest
          const int kk = tid & (EV_KC - 1);
#pragma unroll
          for (int x = 0; x < 4; ++x) {
            const int a = (tid >> 4) + 8 * x;
            cplx v = make_double2(0.0, 0.0);
            if (a0 + a < m && k0 + kk < K) v = A[(long long)(a0 + a) * K + k0 + kk];
            const double sc = (ks && k0 + kk < K) ? wt * ks[k0 + kk] : wt;
            v.x *= sc; v.y *= sc;
            ra[x] = v;
          }
        } else {        // stored K x m, conjugated: a fastest
          const int a = tid & (U1_TILE - 1);
#pragma unroll
          for (int x = 0; x < 4; ++x) {
            const int kk = (tid >> 5) + 4 * x;
            cplx v = make_double2(0.0, 0.0);
            if (a0 + a < m && k0 + kk < K) { v = A[(long long)(k0 + kk) * m + a0 + a]; v.y = -v.y; }
            const double sc = (ks && k0 + kk < K) ? wt * ks[k0 + kk] : wt;
            v.x *= sc; v.y *= sc;
            ra[x] = v;
          }
        }
        // B chunk: 16 (kk) x 32 (b)
        if (!D.opB) {   // stored K x n: b fastest
          const int b = tid & (U1_TILE - 1);
#pragma unroll
          for (int x = 0; x < 4; ++x) {
            const int kk = (tid >> 5) + 4 * x;
            cplx v = make_double2(0.0, 0.0);
            if (b0 + b < n && k0 + kk < K) v = B[(long long)(k0 + kk) * n + b0 + b];
            rb[x] = v;
          }
        } else {        // stored n x K, conjugated: kk fastest
          const int kk = tid & (EV_KC - 1);
#pragma unroll
          for (int x = 0; x < 4; ++x) {
            const int b = (tid >> 4) + 8 * x;
            cplx v = make_double2(0.0, 0.0);
            if (b0 + b < n && k0 + kk < K) { v = B[(long long)(b0 + b) * K + k0 + kk]; v.y = -v.y; }
            rb[x] = v;
          }
        }
        __syncthreads();  // the previous chunk has been consumed
#pragma unroll
        for (int x = 0; x < 4; ++x) {
          if (!D.opA) As[(tid & (EV_KC - 1)) * EV_LD + (tid >> 4) + 8 * x] = ra[x];
          else As[((tid >> 5) + 4 * x) * EV_LD + (tid & (U1_TILE - 1))] = ra[x];
          if (!D.opB) Bs[((tid >> 5) + 4 * x) * EV_LD + (tid & (U1_TILE - 1))] = rb[x];
          else Bs[(tid & (EV_KC - 1)) * EV_LD + (tid >> 4) + 8 * x] = rb[x];
        }
        __syncthreads();
        const int nk = (min(EV_KC, K - k0) + 3) >> 2;
        for (int kq = 0; kq < nk; ++kq) {
          const cplx av = As[(4 * kq + lk) * EV_LD + 8 * warp + lr];
          const double nai = -av.y;
#pragma unroll
          for (int u = 0; u < 4; ++u) {
            const cplx bv = Bs[(4 * kq + lk) * EV_LD + 8 * u + lr];
            dmma(cre[u][0], cre[u][1], av.x, bv.x); dmma(cre[u][0], cre[u][1], nai, bv.y);
            dmma(cim[u][0], cim[u][1], av.x, bv.y); dmma(cim[u][0], cim[u][1], av.y, bv.x);
          }
        }
      }
    }
    __syncthreads();  // before the next tile refills the stages
    const int a = a0 + 8 * warp + lr;
    if (a < m) {
      const double ra_ = D.alpha * (D.rs ? D.rs[a] : 1.0);
#pragma unroll
      for (int u = 0; u < 4; ++u)
#pragma unroll
        for (int x = 0; x < 2; ++x) {
          const int b = b0 + 8 * u + 2 * lk + x;
          if (b < n) {
            const double sc = ra_ * (D.cs ? D.cs[b] : 1.0);
            D.C[(long long)a * n + b] = make_double2(cre[u][x] * sc, cim[u][x] * sc);
          }
        }
    }
  }
}

// Re sum_e T[e] conj(S[e]) over [0, len): K slices, lanes / warps / slices summed in a fixed order (the last CTA adds
// the slice sums), so the result does not depend on timing.
#define EV_DOT_THREADS 256
#define EV_DOT_SLICES 128
__global__ void __launch_bounds__(EV_DOT_THREADS) env_dot_kernel(const cplx* __restrict__ T, const cplx* __restrict__ Sb, long long len,
                                                                 double* part, int* count, double* out) {
  __shared__ double red[EV_DOT_THREADS / 32];
  __shared__ int s_last;
  const int tid = threadIdx.x, K = gridDim.x, j = blockIdx.x;
  const long long e0 = len * j / K, e1 = len * (j + 1) / K;
  double acc = 0.0;
  for (long long e = e0 + tid; e < e1; e += EV_DOT_THREADS) {
    const cplx t = T[e], s = Sb[e];
    acc = fma(t.x, s.x, fma(t.y, s.y, acc));
  }
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) acc += __shfl_xor_sync(0xffffffffu, acc, o);
  if ((tid & 31) == 0) red[tid >> 5] = acc;
  __syncthreads();
  if (tid == 0) {
    double t = 0.0;
    for (int w = 0; w < EV_DOT_THREADS / 32; ++w) t += red[w];
    part[j] = t;
    __threadfence();
    s_last = (atomicAdd(count, 1) == K - 1) ? 1 : 0;
  }
  __syncthreads();
  if (s_last && tid == 0) {
    __threadfence();
    double t = 0.0;
    for (int jj = 0; jj < K; ++jj) t += __ldcg(&part[jj]);
    *out = t;
    *count = 0;
  }
}

// <n_s> = (sum over blocks of (cl - cr) tr(...)) / <psi|psi>,  <psi|psi> = E_M[0]
__global__ void env_finish_kernel(double* out, int M, const cplx* norm) {
  const double inv = 1.0 / norm->x;
  for (int s = threadIdx.x; s < M; s += blockDim.x) out[s] *= inv;
}

namespace {
inline size_t al256(size_t x) { return (x + 255) & ~(size_t)255; }

struct EnvLayout {
  std::vector<long long> Ebase;   // [M+1] element offset of the environments of bond k inside the E store
  std::vector<long long> eoff;    // [(M+1)*NC] offset of sector c inside bond k's environments
  long long Etot = 0, maxE = 0, maxG = 0;
  size_t ndesc = 0, npref = 0;    // descriptors and tile-prefix entries of all launches
  size_t o_desc = 0, o_pref = 0, o_E = 0, o_R = 0, o_T = 0, o_S = 0, o_misc = 0, total = 0;
};

EnvLayout env_layout(int M, int NC, int d, const std::vector<int>& nb, const std::vector<long long>& gused) {
  EnvLayout Y;
  Y.Ebase.resize(M + 1); Y.eoff.assign((size_t)(M + 1) * NC, 0);
  for (int k = 0; k <= M; ++k) {
    Y.Ebase[k] = Y.Etot;
    long long run = 0;
    for (int c = 0; c < NC; ++c) { Y.eoff[(size_t)k * NC + c] = run; const long long n = nb[(size_t)k * NC + c]; run += n * n; }
    Y.Etot += run;
    Y.maxE = std::max(Y.maxE, run);
  }
  for (int s = 0; s < M; ++s) {
    Y.maxG = std::max(Y.maxG, gused[s]);
    size_t nblk = 0, nblk1 = 0, nL = 0, nR = 0;
    for (int cl = 0; cl < NC; ++cl) {
      if (nb[(size_t)s * NC + cl]) ++nL;
      if (nb[(size_t)(s + 1) * NC + cl]) ++nR;
      for (int i = 0; i < d && cl - i >= 0; ++i)
        if (nb[(size_t)s * NC + cl] && nb[(size_t)(s + 1) * NC + cl - i]) { ++nblk; if (i) ++nblk1; }
    }
    // launches of a site: L1 (blocks), L2 (right sectors), R1 (blocks), TT (blocks with i >= 1), R2 (left sectors)
    Y.ndesc += 2 * nblk + nblk1 + nL + nR;
    Y.npref += 2 * nblk + nblk1 + nL + nR + 5;
  }
  size_t o = 0;
  Y.o_desc = o; o = al256(o + Y.ndesc * sizeof(EnvDesc));
  Y.o_pref = o; o = al256(o + Y.npref * sizeof(int));
  Y.o_E = o;    o = al256(o + (size_t)Y.Etot * sizeof(cplx));
  Y.o_R = o;    o = al256(o + (size_t)2 * Y.maxE * sizeof(cplx));
  Y.o_T = o;    o = al256(o + (size_t)Y.maxG * sizeof(cplx));
  Y.o_S = o;    o = al256(o + (size_t)Y.maxG * sizeof(cplx));
  Y.o_misc = o; o = al256(o + (EV_DOT_SLICES + 8) * sizeof(double));
  Y.total = o;
  return Y;
}
}  // namespace

size_t u1_env_scratch_bytes(int M, int NC, int d, const std::vector<int>& nb, const std::vector<long long>& gused) {
  return env_layout(M, NC, d, nb, gused).total;
}

// Host driver: descriptors of all stages from the sector tables, one upload, then the two sweeps.
// nb: [(M+1)*NC] sector sizes; gamoff: [M*NC*d] block offsets of every site; gused: [M] elements used per site.
cudaError_t u1_env_expect_n(const DevState& S, const std::vector<int>& nb, const std::vector<long long>& gamoff,
                            const std::vector<long long>& gused, void* scratch, double* out_dev, const LaunchCfg& L) {
  const int M = S.M, NC = S.NC, d = S.d;
  const EnvLayout Y = env_layout(M, NC, d, nb, gused);
  char* base = (char*)scratch;
  EnvDesc* d_desc = (EnvDesc*)(base + Y.o_desc);
  int* d_pref = (int*)(base + Y.o_pref);
  cplx* Ebuf = (cplx*)(base + Y.o_E);
  cplx* Rbuf = (cplx*)(base + Y.o_R);
  cplx* Tbuf = (cplx*)(base + Y.o_T);
  cplx* Sbuf = (cplx*)(base + Y.o_S);
  double* part = (double*)(base + Y.o_misc);
  int* count = (int*)(part + EV_DOT_SLICES);
  // offsets of the sectors inside lambda^[k]
  std::vector<int> ob((size_t)(M + 1) * NC);
  for (int k = 0; k <= M; ++k) { int run = 0; for (int c = 0; c < NC; ++c) { ob[(size_t)k * NC + c] = run; run += nb[(size_t)k * NC + c]; } }
  auto nK = [&](int k, int c) { return nb[(size_t)k * NC + c]; };
  auto Eptr = [&](int k, int c) { return Ebuf + Y.Ebase[k] + Y.eoff[(size_t)k * NC + c]; };
  auto Rptr = [&](int k, int c) { return Rbuf + (size_t)(k & 1) * Y.maxE + Y.eoff[(size_t)k * NC + c]; };
  auto lamp = [&](int k, int c) { return S.lam + (size_t)k * S.chi + ob[(size_t)k * NC + c]; };
  auto goff = [&](int s, int cl, int i) { return gamoff[((size_t)s * NC + cl) * d + i]; };

  struct Launch { size_t d0, p0; int nd, tiles; };
  std::vector<EnvDesc> descs; descs.reserve(Y.ndesc);
  std::vector<int> prefs; prefs.reserve(Y.npref);
  std::vector<Launch> LA((size_t)M * 5);   // per site: L1, L2, R1, TT, R2
  auto begin_launch = [&](Launch& la) { la.d0 = descs.size(); la.p0 = prefs.size(); la.nd = 0; la.tiles = 0; prefs.push_back(0); };
  auto push = [&](Launch& la, const EnvDesc& D) {
    descs.push_back(D);
    la.tiles += u1_ceil_div(D.m, U1_TILE) * u1_ceil_div(D.n, U1_TILE);
    prefs.push_back(la.tiles);
    ++la.nd;
  };
  EnvDesc Z;
  for (int t = 0; t < EV_MAXTERM; ++t) { Z.A[t] = nullptr; Z.B[t] = nullptr; Z.ks[t] = nullptr; Z.k[t] = 0; Z.w[t] = 1.0; }
  Z.C = nullptr; Z.rs = nullptr; Z.cs = nullptr; Z.alpha = 1.0; Z.m = Z.n = Z.nterm = Z.opA = Z.opB = 0;
  for (int s = 0; s < M; ++s) {
    const cplx* G = S.gam + (size_t)s * S.gcap;
    Launch &l1 = LA[(size_t)s * 5], &l2 = LA[(size_t)s * 5 + 1], &r1 = LA[(size_t)s * 5 + 2], &tt = LA[(size_t)s * 5 + 3], &r2 = LA[(size_t)s * 5 + 4];
    // L1: T_f = E_s[cl] Gamma_f            TT: the same, times the occupation i (only i >= 1)
    begin_launch(l1);
    for (int cl = 0; cl < NC; ++cl) for (int i = 0; i < d && cl - i >= 0; ++i) {
      const int nl = nK(s, cl), nr = nK(s + 1, cl - i);
      if (!nl || !nr) continue;
      EnvDesc D = Z; D.m = nl; D.n = nr; D.nterm = 1; D.A[0] = Eptr(s, cl); D.B[0] = G + goff(s, cl, i); D.k[0] = nl; D.C = Tbuf + goff(s, cl, i);
      push(l1, D);
    }
    begin_launch(tt);
    for (int cl = 0; cl < NC; ++cl) for (int i = 1; i < d && cl - i >= 0; ++i) {
      const int nl = nK(s, cl), nr = nK(s + 1, cl - i);
      if (!nl || !nr) continue;
      EnvDesc D = Z; D.m = nl; D.n = nr; D.nterm = 1; D.A[0] = Eptr(s, cl); D.B[0] = G + goff(s, cl, i); D.k[0] = nl; D.C = Tbuf + goff(s, cl, i);
      D.alpha = (double)i;
      push(tt, D);
    }
    // L2: E_{s+1}[cr] = lam (sum_i Gamma_f^H T_f) lam
    begin_launch(l2);
    for (int cr = 0; cr < NC; ++cr) {
      const int nr = nK(s + 1, cr);
      if (!nr) continue;
      EnvDesc D = Z; D.m = nr; D.n = nr; D.opA = 1; D.C = Eptr(s + 1, cr); D.rs = lamp(s + 1, cr); D.cs = lamp(s + 1, cr);
      for (int i = 0; i < d && cr + i < NC; ++i) {
        const int nl = nK(s, cr + i);
        if (!nl) continue;
        D.A[D.nterm] = G + goff(s, cr + i, i); D.B[D.nterm] = Tbuf + goff(s, cr + i, i); D.k[D.nterm] = nl; ++D.nterm;
      }
      push(l2, D);   // (no term: a sector no block reaches - its environment is zero, and is written as such)
    }
    // R1: S_f = Gamma_f lam R_{s+1}[cr] lam
    begin_launch(r1);
    for (int cl = 0; cl < NC; ++cl) for (int i = 0; i < d && cl - i >= 0; ++i) {
      const int nl = nK(s, cl), nr = nK(s + 1, cl - i);
      if (!nl || !nr) continue;
      EnvDesc D = Z; D.m = nl; D.n = nr; D.nterm = 1; D.A[0] = G + goff(s, cl, i); D.ks[0] = lamp(s + 1, cl - i); D.B[0] = Rptr(s + 1, cl - i);
      D.k[0] = nr; D.cs = lamp(s + 1, cl - i); D.C = Sbuf + goff(s, cl, i);
      push(r1, D);
    }
    // R2: R_s[cl] = sum_i S_f Gamma_f^H
    begin_launch(r2);
    for (int cl = 0; cl < NC; ++cl) {
      const int nl = nK(s, cl);
      if (!nl) continue;
      EnvDesc D = Z; D.m = nl; D.n = nl; D.opB = 1; D.C = Rptr(s, cl);
      for (int i = 0; i < d && cl - i >= 0; ++i) {
        const int nr = nK(s + 1, cl - i);
        if (!nr) continue;
        D.A[D.nterm] = Sbuf + goff(s, cl, i); D.B[D.nterm] = G + goff(s, cl, i); D.k[D.nterm] = nr; ++D.nterm;
      }
      push(r2, D);   // (no term: a dead-end sector, left behind by a truncation - zero environment)
    }
  }
  cudaError_t err;
  if ((err = cudaMemcpyAsync(d_desc, descs.data(), descs.size() * sizeof(EnvDesc), cudaMemcpyHostToDevice, L.stream)) != cudaSuccess) return err;
  if ((err = cudaMemcpyAsync(d_pref, prefs.data(), prefs.size() * sizeof(int), cudaMemcpyHostToDevice, L.stream)) != cudaSuccess) return err;
  if ((err = cudaMemsetAsync(Ebuf, 0, (size_t)Y.Etot * sizeof(cplx), L.stream)) != cudaSuccess) return err;
  if ((err = cudaMemsetAsync(Rbuf, 0, (size_t)2 * Y.maxE * sizeof(cplx), L.stream)) != cudaSuccess) return err;
  if ((err = cudaMemsetAsync(part, 0, (EV_DOT_SLICES + 8) * sizeof(double), L.stream)) != cudaSuccess) return err;
  const cplx one = make_double2(1.0, 0.0);
  if ((err = cudaMemcpyAsync(Eptr(0, S.N), &one, sizeof(cplx), cudaMemcpyHostToDevice, L.stream)) != cudaSuccess) return err;
  if ((err = cudaMemcpyAsync(Rptr(M, 0), &one, sizeof(cplx), cudaMemcpyHostToDevice, L.stream)) != cudaSuccess) return err;
  // the host vectors must outlive the asynchronous copies out of pageable memory: those are staged by the runtime before
  // the call returns, so nothing more is needed here
  auto run = [&](const Launch& la) {
    if (la.tiles == 0) return;
    L.prof->begin(U1_ST_READOUT, L.stream);
    env_gemm_kernel<<<std::min(la.tiles, L.sms * 8), EV_THREADS, 0, L.stream>>>(d_desc + la.d0, d_pref + la.p0, la.nd);
    L.prof->end(L.stream);
    ++*L.launches;
  };
  for (int s = 0; s < M; ++s) { run(LA[(size_t)s * 5]); run(LA[(size_t)s * 5 + 1]); }
  for (int s = M - 1; s >= 0; --s) {
    run(LA[(size_t)s * 5 + 2]);
    if ((err = cudaMemsetAsync(Tbuf, 0, (size_t)gused[s] * sizeof(cplx), L.stream)) != cudaSuccess) return err;
    run(LA[(size_t)s * 5 + 3]);
    L.prof->begin(U1_ST_READOUT, L.stream);
    env_dot_kernel<<<EV_DOT_SLICES, EV_DOT_THREADS, 0, L.stream>>>(Tbuf, Sbuf, gused[s], part, count, out_dev + s);
    L.prof->end(L.stream);
    ++*L.launches;
    run(LA[(size_t)s * 5 + 4]);
  }
  env_finish_kernel<<<1, 256, 0, L.stream>>>(out_dev, M, Eptr(M, 0));
  ++*L.launches;
  return cudaGetLastError();
}

// ---------------------------------------------------------------------------------------------------------------------
// Two-point function <psi|n_j n_k|psi> / <psi|psi>, j <= k: the same sweeps with the weight
// (c_l - c_r) inserted into the transfer step of site j; F is the left environment that carries the insertion.
//   F_{j+1}[cr] = sum_cl (cl - cr) A^H E_j[cl] A,   F_{s+1}[cr] = sum_cl A^H F_s[cl] A  (s > j)
//   value = sum (cl - cr) tr(A^H F_k[cl] A R_{k+1}[cr])      (j < k;  (cl - cr)^2 and E_k for j == k)
//   norm  = sum tr(A^H E_k[cl] A R_{k+1}[cr])
__global__ void env_ratio_kernel(double* out, const double* val, const double* norm) { *out = *val / *norm; }

namespace {
struct NNLayout { long long maxE = 0, maxG = 0; size_t ndesc = 0, npref = 0, o_desc = 0, o_pref = 0, o_E = 0, o_F = 0, o_R = 0, o_T = 0, o_S = 0, o_misc = 0, total = 0; };
NNLayout nn_layout(int M, int NC, int d, const std::vector<int>& nb, const std::vector<long long>& gused) {
  NNLayout Y;
  size_t per_site = 0;
  for (int k = 0; k <= M; ++k) {
    long long run = 0; size_t nsec = 0;
    for (int c = 0; c < NC; ++c) { const long long n = nb[(size_t)k * NC + c]; run += n * n; nsec += n > 0; }
    Y.maxE = std::max(Y.maxE, run);
    per_site = std::max(per_site, nsec);
  }
  size_t maxblk = 0;
  for (int s = 0; s < M; ++s) {
    Y.maxG = std::max(Y.maxG, gused[s]);
    size_t nblk = 0;
    for (int cl = 0; cl < NC; ++cl) for (int i = 0; i < d && cl - i >= 0; ++i)
      if (nb[(size_t)s * NC + cl] && nb[(size_t)(s + 1) * NC + cl - i]) ++nblk;
    maxblk = std::max(maxblk, nblk);
  }
  Y.ndesc = (size_t)(M + 2) * (2 * maxblk + 3 * per_site + 2);   // generous: at most 2 block launches + 3 sector launches per site
  Y.npref = Y.ndesc + (size_t)(M + 2) * 6;
  size_t o = 0;
  Y.o_desc = o; o = al256(o + Y.ndesc * sizeof(EnvDesc));
  Y.o_pref = o; o = al256(o + Y.npref * sizeof(int));
  Y.o_E = o;    o = al256(o + (size_t)2 * Y.maxE * sizeof(cplx));
  Y.o_F = o;    o = al256(o + (size_t)2 * Y.maxE * sizeof(cplx));
  Y.o_R = o;    o = al256(o + (size_t)2 * Y.maxE * sizeof(cplx));
  Y.o_T = o;    o = al256(o + (size_t)Y.maxG * sizeof(cplx));
  Y.o_S = o;    o = al256(o + (size_t)Y.maxG * sizeof(cplx));
  Y.o_misc = o; o = al256(o + (EV_DOT_SLICES + 8) * sizeof(double));
  Y.total = o;
  return Y;
}
}  // namespace

size_t u1_env_nn_scratch_bytes(int M, int NC, int d, const std::vector<int>& nb, const std::vector<long long>& gused) {
  return nn_layout(M, NC, d, nb, gused).total;
}

cudaError_t u1_env_expect_nn(const DevState& S, const std::vector<int>& nb, const std::vector<long long>& gamoff,
                             const std::vector<long long>& gused, int j, int k, void* scratch, double* out_dev, const LaunchCfg& L) {
  const int M = S.M, NC = S.NC, d = S.d;
  const NNLayout Y = nn_layout(M, NC, d, nb, gused);
  char* base = (char*)scratch;
  EnvDesc* d_desc = (EnvDesc*)(base + Y.o_desc);
  int* d_pref = (int*)(base + Y.o_pref);
  cplx* Ebuf = (cplx*)(base + Y.o_E);
  cplx* Fbuf = (cplx*)(base + Y.o_F);
  cplx* Rbuf = (cplx*)(base + Y.o_R);
  cplx* Tbuf = (cplx*)(base + Y.o_T);
  cplx* Sbuf = (cplx*)(base + Y.o_S);
  double* part = (double*)(base + Y.o_misc);
  int* count = (int*)(part + EV_DOT_SLICES);
  double* scal = part + EV_DOT_SLICES + 2;   // [0] value, [1] norm
  std::vector<int> ob((size_t)(M + 1) * NC);
  std::vector<long long> eoff((size_t)(M + 1) * NC);
  for (int b = 0; b <= M; ++b) {
    int run = 0; long long er = 0;
    for (int c = 0; c < NC; ++c) { ob[(size_t)b * NC + c] = run; eoff[(size_t)b * NC + c] = er; const long long n = nb[(size_t)b * NC + c]; run += (int)n; er += n * n; }
  }
  auto nK = [&](int b, int c) { return nb[(size_t)b * NC + c]; };
  auto envp = [&](cplx* buf, int b, int c) { return buf + (size_t)(b & 1) * Y.maxE + eoff[(size_t)b * NC + c]; };
  auto lamp = [&](int b, int c) { return S.lam + (size_t)b * S.chi + ob[(size_t)b * NC + c]; };
  auto goff = [&](int s, int cl, int i) { return gamoff[((size_t)s * NC + cl) * d + i]; };
  struct Launch { size_t d0, p0; int nd, tiles; };
  std::vector<EnvDesc> descs;
  std::vector<int> prefs;
  std::vector<Launch> order;
  EnvDesc Z;
  for (int t = 0; t < EV_MAXTERM; ++t) { Z.A[t] = nullptr; Z.B[t] = nullptr; Z.ks[t] = nullptr; Z.k[t] = 0; Z.w[t] = 1.0; }
  Z.C = nullptr; Z.rs = nullptr; Z.cs = nullptr; Z.alpha = 1.0; Z.m = Z.n = Z.nterm = Z.opA = Z.opB = 0;
  Launch cur;
  auto begin = [&]() { cur.d0 = descs.size(); cur.p0 = prefs.size(); cur.nd = 0; cur.tiles = 0; prefs.push_back(0); };
  auto push = [&](const EnvDesc& D) { descs.push_back(D); cur.tiles += u1_ceil_div(D.m, U1_TILE) * u1_ceil_div(D.n, U1_TILE); prefs.push_back(cur.tiles); ++cur.nd; };
  auto end = [&]() { order.push_back(cur); };
  // dst_f = alpha(i) env[cl] Gamma_f for the blocks of site s (alpha == 0: skipped)
  auto mkT = [&](int s, cplx* env, cplx* dst, int power) {
    begin();
    const cplx* G = S.gam + (size_t)s * S.gcap;
    for (int cl = 0; cl < NC; ++cl) for (int i = 0; i < d && cl - i >= 0; ++i) {
      const int nl = nK(s, cl), nr = nK(s + 1, cl - i);
      if (!nl || !nr) continue;
      const double al = power == 0 ? 1.0 : power == 1 ? (double)i : (double)i * i;
      if (al == 0.0) continue;
      EnvDesc D = Z; D.m = nl; D.n = nr; D.nterm = 1; D.A[0] = envp(env, s, cl); D.B[0] = G + goff(s, cl, i); D.k[0] = nl; D.C = dst + goff(s, cl, i); D.alpha = al;
      push(D);
    }
    end();
  };
  // env'[cr] = lam (sum_i w_i Gamma_f^H src_f) lam for the sectors of bond s+1 (weighted: w_i = i)
  auto mkL2 = [&](int s, const cplx* src, cplx* env, bool weighted) {
    begin();
    const cplx* G = S.gam + (size_t)s * S.gcap;
    for (int cr = 0; cr < NC; ++cr) {
      const int nr = nK(s + 1, cr);
      if (!nr) continue;
      EnvDesc D = Z; D.m = nr; D.n = nr; D.opA = 1; D.C = envp(env, s + 1, cr); D.rs = lamp(s + 1, cr); D.cs = lamp(s + 1, cr);
      for (int i = weighted ? 1 : 0; i < d && cr + i < NC; ++i) {
        const int nl = nK(s, cr + i);
        if (!nl) continue;
        D.A[D.nterm] = G + goff(s, cr + i, i); D.B[D.nterm] = src + goff(s, cr + i, i); D.k[D.nterm] = nl; D.w[D.nterm] = weighted ? (double)i : 1.0; ++D.nterm;
      }
      push(D);
    }
    end();
  };
  auto mkR1 = [&](int s) {   // S_f = Gamma_f lam R_{s+1}[cr] lam
    begin();
    const cplx* G = S.gam + (size_t)s * S.gcap;
    for (int cl = 0; cl < NC; ++cl) for (int i = 0; i < d && cl - i >= 0; ++i) {
      const int nl = nK(s, cl), nr = nK(s + 1, cl - i);
      if (!nl || !nr) continue;
      EnvDesc D = Z; D.m = nl; D.n = nr; D.nterm = 1; D.A[0] = G + goff(s, cl, i); D.ks[0] = lamp(s + 1, cl - i); D.B[0] = envp(Rbuf, s + 1, cl - i);
      D.k[0] = nr; D.cs = lamp(s + 1, cl - i); D.C = Sbuf + goff(s, cl, i);
      push(D);
    }
    end();
  };
  auto mkR2 = [&](int s) {   // R_s[cl] = sum_i S_f Gamma_f^H
    begin();
    const cplx* G = S.gam + (size_t)s * S.gcap;
    for (int cl = 0; cl < NC; ++cl) {
      const int nl = nK(s, cl);
      if (!nl) continue;
      EnvDesc D = Z; D.m = nl; D.n = nl; D.opB = 1; D.C = envp(Rbuf, s, cl);
      for (int i = 0; i < d && cl - i >= 0; ++i) {
        const int nr = nK(s + 1, cl - i);
        if (!nr) continue;
        D.A[D.nterm] = Sbuf + goff(s, cl, i); D.B[D.nterm] = G + goff(s, cl, i); D.k[D.nterm] = nr; ++D.nterm;
      }
      push(D);
    }
    end();
  };
  // launch order; entries of `order` are consumed in this order below, interleaved with the memsets and dots
  for (int s = 0; s < k; ++s) {
    mkT(s, Ebuf, Tbuf, 0); mkL2(s, Tbuf, Ebuf, false);
    if (s == j) mkL2(s, Tbuf, Fbuf, true);
    else if (s > j) { mkT(s, Fbuf, Sbuf, 0); mkL2(s, Sbuf, Fbuf, false); }
  }
  for (int s = M - 1; s > k; --s) { mkR1(s); mkR2(s); }
  mkR1(k);
  mkT(k, Ebuf, Tbuf, 0);                              // norm
  if (j < k) mkT(k, Fbuf, Tbuf, 1); else mkT(k, Ebuf, Tbuf, 2);   // value
  if (descs.size() > Y.ndesc || prefs.size() > Y.npref) return cudaErrorInvalidValue;
  cudaError_t err;
  if ((err = cudaMemcpyAsync(d_desc, descs.data(), descs.size() * sizeof(EnvDesc), cudaMemcpyHostToDevice, L.stream)) != cudaSuccess) return err;
  if ((err = cudaMemcpyAsync(d_pref, prefs.data(), prefs.size() * sizeof(int), cudaMemcpyHostToDevice, L.stream)) != cudaSuccess) return err;
  if ((err = cudaMemsetAsync(Ebuf, 0, (size_t)2 * Y.maxE * sizeof(cplx), L.stream)) != cudaSuccess) return err;
  if ((err = cudaMemsetAsync(Fbuf, 0, (size_t)2 * Y.maxE * sizeof(cplx), L.stream)) != cudaSuccess) return err;
  if ((err = cudaMemsetAsync(Rbuf, 0, (size_t)2 * Y.maxE * sizeof(cplx), L.stream)) != cudaSuccess) return err;
  if ((err = cudaMemsetAsync(part, 0, (EV_DOT_SLICES + 8) * sizeof(double), L.stream)) != cudaSuccess) return err;
  const cplx one = make_double2(1.0, 0.0);
  if ((err = cudaMemcpyAsync(envp(Ebuf, 0, S.N), &one, sizeof(cplx), cudaMemcpyHostToDevice, L.stream)) != cudaSuccess) return err;
  if ((err = cudaMemcpyAsync(envp(Rbuf, M, 0), &one, sizeof(cplx), cudaMemcpyHostToDevice, L.stream)) != cudaSuccess) return err;
  auto run = [&](const Launch& la) {
    if (la.tiles == 0) return;
    L.prof->begin(U1_ST_READOUT, L.stream);
    env_gemm_kernel<<<std::min(la.tiles, L.sms * 8), EV_THREADS, 0, L.stream>>>(d_desc + la.d0, d_pref + la.p0, la.nd);
    L.prof->end(L.stream);
    ++*L.launches;
  };
  const size_t n_final = 3;   // R1(k), T(norm), T(value)
  for (size_t q = 0; q + n_final < order.size(); ++q) run(order[q]);
  const size_t q0 = order.size() - n_final;
  run(order[q0]);                                       // S_f at site k
  for (int pass = 0; pass < 2; ++pass) {                // norm, then value
    if ((err = cudaMemsetAsync(Tbuf, 0, (size_t)gused[k] * sizeof(cplx), L.stream)) != cudaSuccess) return err;
    run(order[q0 + 1 + pass]);
    env_dot_kernel<<<EV_DOT_SLICES, EV_DOT_THREADS, 0, L.stream>>>(Tbuf, Sbuf, gused[k], part, count, scal + (pass == 0 ? 1 : 0));
    ++*L.launches;
  }
  env_ratio_kernel<<<1, 1, 0, L.stream>>>(out_dev, scal, scal + 1);
  ++*L.launches;
  return cudaGetLastError();
}

// ---------------------------------------------------------------------------------------------------------------------
// Fock-pattern sampling (the output distribution over occupation patterns; state
// of Eq.15): patterns drawn from |<n|psi>|^2 / <psi|psi> site by site, exactly, for whatever Gamma, lambda the
// handle holds.  All right environments R_s[cl] = sum_cr A R_{s+1}[cr] A^H are built once by the grouped GEMMs above and
// kept; then one launch per site advances every sample: a sample at bond s with charge c and boundary row vector v takes
// occupation i with weight p_i = w_i R_{s+1}[c - i] w_i^H, w_i = v Gamma^[s][c, c - i] diag(lambda^[s+1][c - i]), by
// inverse CDF on the uniform number the caller passed for (sample, site); v <- w_i / sqrt(p_i), c <- c - i.
// One CTA per sample; the vector-matrix products split the inner index over the 8 warps and the output index over the
// lanes (coalesced rows), partial sums added in warp order: results do not depend on timing.
#define FS_THREADS 256
#define FS_WARPS (FS_THREADS / 32)
#define FS_BC 256   // output columns per pass (8 per lane)

// out[b] = sc[b] * sum_a v[a] Mt[a * n_out + b]  (store != nullptr), or the return value (valid in every thread)
// Re sum_b (sum_a v[a] Mt[a * n_out + b]) conj(wref[b])  (store == nullptr)
__device__ double fs_vecmat(const cplx* __restrict__ v, int n_in, const cplx* __restrict__ Mt, int n_out, const double* __restrict__ sc,
                            cplx* store, const cplx* wref, cplx* part, double* red) {
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  const int a0 = (int)((long long)n_in * warp / FS_WARPS), a1 = (int)((long long)n_in * (warp + 1) / FS_WARPS);
  double dacc = 0.0;
  for (int b0 = 0; b0 < n_out; b0 += FS_BC) {
    double ar[FS_BC / 32], ai[FS_BC / 32];
#pragma unroll
    for (int x = 0; x < FS_BC / 32; ++x) { ar[x] = 0.0; ai[x] = 0.0; }
    for (int a = a0; a < a1; ++a) {
      const cplx va = v[a];
      const cplx* row = Mt + (long long)a * n_out + b0 + lane;
#pragma unroll
      for (int x = 0; x < FS_BC / 32; ++x) {
        if (b0 + lane + 32 * x < n_out) {
          const cplx g = row[32 * x];
          ar[x] = fma(va.x, g.x, fma(-va.y, g.y, ar[x]));
          ai[x] = fma(va.x, g.y, fma(va.y, g.x, ai[x]));
        }
      }
    }
#pragma unroll
    for (int x = 0; x < FS_BC / 32; ++x) part[warp * FS_BC + lane + 32 * x] = make_double2(ar[x], ai[x]);
    __syncthreads();
    if (b0 + tid < n_out) {   // FS_THREADS == FS_BC: one output column per thread
      double tr = 0.0, ti = 0.0;
#pragma unroll
      for (int w = 0; w < FS_WARPS; ++w) { const cplx q = part[w * FS_BC + tid]; tr += q.x; ti += q.y; }
      if (store) {
        const double s = sc ? sc[b0 + tid] : 1.0;
        store[b0 + tid] = make_double2(tr * s, ti * s);
      } else {
        const cplx r = wref[b0 + tid];
        dacc = fma(tr, r.x, fma(ti, r.y, dacc));
      }
    }
    __syncthreads();
  }
  if (store) return 0.0;
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) dacc += __shfl_xor_sync(0xffffffffu, dacc, o);
  if (lane == 0) red[warp] = dacc;
  __syncthreads();
  double t = 0.0;
#pragma unroll
  for (int w = 0; w < FS_WARPS; ++w) t += red[w];
  __syncthreads();
  return t;
}
static_assert(FS_THREADS == FS_BC, "fs_vecmat: one output column per thread");

__global__ void __launch_bounds__(FS_THREADS) fock_step_kernel(DevState S, int s, const cplx* __restrict__ Rall, const long long* __restrict__ roff,
                                                               const double* __restrict__ u, const cplx* __restrict__ vcur, cplx* vnext, cplx* wbuf,
                                                               int* cs, int* pat, double* logp, int maxn) {
  __shared__ __align__(16) cplx part[FS_WARPS * FS_BC];
  __shared__ double red[FS_WARPS];
  __shared__ double s_p[EV_MAXTERM];
  __shared__ int s_pick;
  __shared__ double s_scale;
  const int b = blockIdx.x, tid = threadIdx.x, NC = S.NC, d = S.d, M = S.M;
  const int c = cs[b];
  const int* nbL = S.nb + (long long)s * NC;
  const int* nbR = S.nb + (long long)(s + 1) * NC;
  const int nl = nbL[c];
  const cplx* v = vcur + (long long)b * maxn;
  const cplx* gam = S.gam + (long long)s * S.gcap;
  const long long* goff = S.gamoff + (long long)s * NC * d;
  for (int i = 0; i < d; ++i) {
    const int cr = c - i;
    double p = 0.0;
    const int nr = cr >= 0 ? nbR[cr] : 0;
    if (nr > 0 && nl > 0) {   // uniform over the CTA
      cplx* w = wbuf + ((long long)b * d + i) * maxn;
      fs_vecmat(v, nl, gam + goff[c * d + i], nr, S.lam + (long long)(s + 1) * S.chi + S.ob[(long long)(s + 1) * NC + cr], w, nullptr, part, red);
      __syncthreads();   // w (global) is read back by other threads of the CTA
      p = fs_vecmat(w, nr, Rall + roff[(long long)(s + 1) * NC + cr], nr, nullptr, nullptr, w, part, red);
    }
    if (tid == 0) s_p[i] = p;
  }
  __syncthreads();
  if (tid == 0) {
    double tot = 0.0;
    for (int i = 0; i < d; ++i) tot += s_p[i];
    const double target = u[(long long)b * M + s] * tot;
    double cum = 0.0;
    int pick = -1, last = 0;
    for (int i = 0; i < d; ++i) {
      cum += s_p[i];
      if (s_p[i] > 0.0) { last = i; if (pick < 0 && target < cum) pick = i; }
    }
    if (pick < 0) pick = last;   // rounding at the top of the CDF
    pat[(long long)b * M + s] = pick;
    logp[b] += log(s_p[pick] / tot);
    cs[b] = c - pick;
    s_pick = pick;
    s_scale = rsqrt(s_p[pick]);
  }
  __syncthreads();
  const int pick = s_pick;
  const int nrp = (c - pick >= 0) ? nbR[c - pick] : 0;
  const double sc = s_scale;
  const cplx* w = wbuf + ((long long)b * d + pick) * maxn;
  cplx* vn = vnext + (long long)b * maxn;
  for (int x = tid; x < nrp; x += FS_THREADS) { const cplx q = w[x]; vn[x] = make_double2(q.x * sc, q.y * sc); }
}

__global__ void fock_init_kernel(int B, int N, int maxn, cplx* vcur, int* cs, double* logp) {
  const int b = blockIdx.x * blockDim.x + threadIdx.x;
  if (b >= B) return;
  vcur[(long long)b * maxn] = make_double2(1.0, 0.0);
  cs[b] = N;
  logp[b] = 0.0;
}

namespace {
struct FockLayout {
  EnvLayout E;          // Ebase / eoff / Etot / maxG (its own offsets are not used here)
  int maxn = 1;
  size_t ndesc = 0, npref = 0;
  size_t o_desc = 0, o_pref = 0, o_R = 0, o_S = 0, o_roff = 0, o_u = 0, o_pat = 0, o_logp = 0, o_cs = 0, o_v0 = 0, o_v1 = 0, o_w = 0, total = 0;
};
FockLayout fock_layout(int M, int NC, int d, const std::vector<int>& nb, const std::vector<long long>& gused, int B) {
  FockLayout Y;
  Y.E = env_layout(M, NC, d, nb, gused);
  for (size_t x = 0; x < nb.size(); ++x) Y.maxn = std::max(Y.maxn, nb[x]);
  for (int s = 0; s < M; ++s) {
    size_t nblk = 0, nL = 0;
    for (int cl = 0; cl < NC; ++cl) {
      if (nb[(size_t)s * NC + cl]) ++nL;
      for (int i = 0; i < d && cl - i >= 0; ++i)
        if (nb[(size_t)s * NC + cl] && nb[(size_t)(s + 1) * NC + cl - i]) ++nblk;
    }
    Y.ndesc += nblk + nL;
    Y.npref += nblk + nL + 2;
  }
  size_t o = 0;
  Y.o_desc = o; o = al256(o + Y.ndesc * sizeof(EnvDesc));
  Y.o_pref = o; o = al256(o + Y.npref * sizeof(int));
  Y.o_R = o;    o = al256(o + (size_t)Y.E.Etot * sizeof(cplx));
  Y.o_S = o;    o = al256(o + (size_t)Y.E.maxG * sizeof(cplx));
  Y.o_roff = o; o = al256(o + (size_t)(M + 1) * NC * sizeof(long long));
  Y.o_u = o;    o = al256(o + (size_t)B * M * sizeof(double));
  Y.o_pat = o;  o = al256(o + (size_t)B * M * sizeof(int));
  Y.o_logp = o; o = al256(o + (size_t)B * sizeof(double));
  Y.o_cs = o;   o = al256(o + (size_t)B * sizeof(int));
  Y.o_v0 = o;   o = al256(o + (size_t)B * Y.maxn * sizeof(cplx));
  Y.o_v1 = o;   o = al256(o + (size_t)B * Y.maxn * sizeof(cplx));
  Y.o_w = o;    o = al256(o + (size_t)B * d * Y.maxn * sizeof(cplx));
  Y.total = o;
  return Y;
}
}  // namespace

size_t u1_env_sample_scratch_bytes(int M, int NC, int d, const std::vector<int>& nb, const std::vector<long long>& gused, int B) {
  return fock_layout(M, NC, d, nb, gused, B).total;
}

// Host driver.  u_host: HOST [B * M] uniform numbers in [0, 1); pat_host: HOST int32 [B * M]; logp_host: HOST [B] (ln of
// the probability of the drawn pattern).  Everything is enqueued on L.stream; the caller synchronises.
cudaError_t u1_env_sample_fock(const DevState& S, const std::vector<int>& nb, const std::vector<long long>& gamoff,
                               const std::vector<long long>& gused, int B, const double* u_host, int* pat_host, double* logp_host,
                               void* scratch, const LaunchCfg& L) {
  const int M = S.M, NC = S.NC, d = S.d;
  const FockLayout Y = fock_layout(M, NC, d, nb, gused, B);
  char* base = (char*)scratch;
  EnvDesc* d_desc = (EnvDesc*)(base + Y.o_desc);
  int* d_pref = (int*)(base + Y.o_pref);
  cplx* Rall = (cplx*)(base + Y.o_R);
  cplx* Sbuf = (cplx*)(base + Y.o_S);
  long long* d_roff = (long long*)(base + Y.o_roff);
  double* d_u = (double*)(base + Y.o_u);
  int* d_pat = (int*)(base + Y.o_pat);
  double* d_logp = (double*)(base + Y.o_logp);
  int* d_cs = (int*)(base + Y.o_cs);
  cplx* v0 = (cplx*)(base + Y.o_v0);
  cplx* v1 = (cplx*)(base + Y.o_v1);
  cplx* wbuf = (cplx*)(base + Y.o_w);
  std::vector<int> ob((size_t)(M + 1) * NC);
  std::vector<long long> roff((size_t)(M + 1) * NC);
  for (int k = 0; k <= M; ++k) {
    int run = 0;
    for (int c = 0; c < NC; ++c) {
      ob[(size_t)k * NC + c] = run; run += nb[(size_t)k * NC + c];
      roff[(size_t)k * NC + c] = Y.E.Ebase[k] + Y.E.eoff[(size_t)k * NC + c];
    }
  }
  auto nK = [&](int k, int c) { return nb[(size_t)k * NC + c]; };
  auto Rptr = [&](int k, int c) { return Rall + roff[(size_t)k * NC + c]; };
  auto lamp = [&](int k, int c) { return S.lam + (size_t)k * S.chi + ob[(size_t)k * NC + c]; };
  auto goff = [&](int s, int cl, int i) { return gamoff[((size_t)s * NC + cl) * d + i]; };
  struct Launch { size_t d0, p0; int nd, tiles; };
  std::vector<EnvDesc> descs; descs.reserve(Y.ndesc);
  std::vector<int> prefs; prefs.reserve(Y.npref);
  std::vector<Launch> LA((size_t)M * 2);   // per site: R1, R2
  auto begin_launch = [&](Launch& la) { la.d0 = descs.size(); la.p0 = prefs.size(); la.nd = 0; la.tiles = 0; prefs.push_back(0); };
  auto push = [&](Launch& la, const EnvDesc& D) {
    descs.push_back(D);
    la.tiles += u1_ceil_div(D.m, U1_TILE) * u1_ceil_div(D.n, U1_TILE);
    prefs.push_back(la.tiles);
    ++la.nd;
  };
  EnvDesc Z;
  for (int t = 0; t < EV_MAXTERM; ++t) { Z.A[t] = nullptr; Z.B[t] = nullptr; Z.ks[t] = nullptr; Z.k[t] = 0; Z.w[t] = 1.0; }
  Z.C = nullptr; Z.rs = nullptr; Z.cs = nullptr; Z.alpha = 1.0; Z.m = Z.n = Z.nterm = Z.opA = Z.opB = 0;
  for (int s = 0; s < M; ++s) {
    const cplx* G = S.gam + (size_t)s * S.gcap;
    Launch &r1 = LA[(size_t)s * 2], &r2 = LA[(size_t)s * 2 + 1];
    begin_launch(r1);   // S_f = Gamma_f lam R_{s+1}[cr] lam
    for (int cl = 0; cl < NC; ++cl) for (int i = 0; i < d && cl - i >= 0; ++i) {
      const int nl = nK(s, cl), nr = nK(s + 1, cl - i);
      if (!nl || !nr) continue;
      EnvDesc D = Z; D.m = nl; D.n = nr; D.nterm = 1; D.A[0] = G + goff(s, cl, i); D.ks[0] = lamp(s + 1, cl - i); D.B[0] = Rptr(s + 1, cl - i);
      D.k[0] = nr; D.cs = lamp(s + 1, cl - i); D.C = Sbuf + goff(s, cl, i);
      push(r1, D);
    }
    begin_launch(r2);   // R_s[cl] = sum_i S_f Gamma_f^H
    for (int cl = 0; cl < NC; ++cl) {
      const int nl = nK(s, cl);
      if (!nl) continue;
      EnvDesc D = Z; D.m = nl; D.n = nl; D.opB = 1; D.C = Rptr(s, cl);
      for (int i = 0; i < d && cl - i >= 0; ++i) {
        const int nr = nK(s + 1, cl - i);
        if (!nr) continue;
        D.A[D.nterm] = Sbuf + goff(s, cl, i); D.B[D.nterm] = G + goff(s, cl, i); D.k[D.nterm] = nr; ++D.nterm;
      }
      push(r2, D);   // (no term: a dead-end sector - zero environment, no sample can enter it)
    }
  }
  if (descs.size() > Y.ndesc || prefs.size() > Y.npref) return cudaErrorInvalidValue;
  cudaError_t err;
  if ((err = cudaMemcpyAsync(d_desc, descs.data(), descs.size() * sizeof(EnvDesc), cudaMemcpyHostToDevice, L.stream)) != cudaSuccess) return err;
  if ((err = cudaMemcpyAsync(d_pref, prefs.data(), prefs.size() * sizeof(int), cudaMemcpyHostToDevice, L.stream)) != cudaSuccess) return err;
  if ((err = cudaMemcpyAsync(d_roff, roff.data(), roff.size() * sizeof(long long), cudaMemcpyHostToDevice, L.stream)) != cudaSuccess) return err;
  if ((err = cudaMemcpyAsync(d_u, u_host, (size_t)B * M * sizeof(double), cudaMemcpyHostToDevice, L.stream)) != cudaSuccess) return err;
  if ((err = cudaMemsetAsync(Rall, 0, (size_t)Y.E.Etot * sizeof(cplx), L.stream)) != cudaSuccess) return err;
  const cplx one = make_double2(1.0, 0.0);
  if ((err = cudaMemcpyAsync(Rptr(M, 0), &one, sizeof(cplx), cudaMemcpyHostToDevice, L.stream)) != cudaSuccess) return err;
  auto run = [&](const Launch& la) {
    if (la.tiles == 0) return;
    L.prof->begin(U1_ST_READOUT, L.stream);
    env_gemm_kernel<<<std::min(la.tiles, L.sms * 8), EV_THREADS, 0, L.stream>>>(d_desc + la.d0, d_pref + la.p0, la.nd);
    L.prof->end(L.stream);
    ++*L.launches;
  };
  for (int s = M - 1; s >= 0; --s) { run(LA[(size_t)s * 2]); run(LA[(size_t)s * 2 + 1]); }
  fock_init_kernel<<<u1_ceil_div(B, 256), 256, 0, L.stream>>>(B, S.N, Y.maxn, v0, d_cs, d_logp);
  ++*L.launches;
  cplx *vc = v0, *vn = v1;
  for (int s = 0; s < M; ++s) {
    L.prof->begin(U1_ST_READOUT, L.stream);
    fock_step_kernel<<<B, FS_THREADS, 0, L.stream>>>(S, s, Rall, d_roff, d_u, vc, vn, wbuf, d_cs, d_pat, d_logp, Y.maxn);
    L.prof->end(L.stream);
    ++*L.launches;
    std::swap(vc, vn);
  }
  if ((err = cudaGetLastError()) != cudaSuccess) return err;
  if ((err = cudaMemcpyAsync(pat_host, d_pat, (size_t)B * M * sizeof(int), cudaMemcpyDeviceToHost, L.stream)) != cudaSuccess) return err;
  return cudaMemcpyAsync(logp_host, d_logp, (size_t)B * sizeof(double), cudaMemcpyDeviceToHost, L.stream);
}
