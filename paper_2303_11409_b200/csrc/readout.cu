// readout.cu — step a6 (canonical-form readouts, SURVEY §8(c) "Readouts"; Eq.10/15 canonical form)
// and the small state-maintenance kernels (product state, block-offset rebuild after an import).
#include "common.cuh"

#define RD_THREADS 256

__device__ __forceinline__ double block_sum(double v, double* sh) {
  const int tid = threadIdx.x;
  sh[tid] = v;
  __syncthreads();
  for (int o = RD_THREADS / 2; o > 0; o >>= 1) {
    if (tid < o) sh[tid] += sh[tid + o];
    __syncthreads();
  }
  const double r = sh[0];
  __syncthreads();
  return r;
}

// <n_s> = sum_{cl,cr} (cl - cr) sum_{a,b} lamL[cl]_a^2 |Gamma[cl,cr]_ab|^2 lamR[cr]_b^2 ; one CTA per site
__global__ void __launch_bounds__(RD_THREADS) expect_n_kernel(DevState S, double* out) {
  __shared__ double sh[RD_THREADS];
  const int s = blockIdx.x, NC = S.NC, d = S.d;
  const int* nbL = S.nb + (long long)s * NC;
  const int* nbR = S.nb + (long long)(s + 1) * NC;
  double acc = 0.0;
  for (int cl = 0; cl < NC; ++cl) {
    const int nl = nbL[cl];
    if (nl == 0) continue;
    const double* lamL = S.lam + (long long)s * S.chi + S.ob[(long long)s * NC + cl];
    for (int i = 1; i < d && cl - i >= 0; ++i) {  // occupation i = 0 contributes nothing
      const int cr = cl - i, nr = nbR[cr];
      if (nr == 0) continue;
      const double* lamR = S.lam + (long long)(s + 1) * S.chi + S.ob[(long long)(s + 1) * NC + cr];
      const cplx* Gm = S.gam + (long long)s * S.gcap + S.gamoff[((long long)s * NC + cl) * d + i];
      double part = 0.0;
      for (long long idx = threadIdx.x; idx < (long long)nl * nr; idx += RD_THREADS) {
        const int a = (int)(idx / nr), b = (int)(idx % nr);
        const cplx v = Gm[idx];
        const double la = lamL[a], lb = lamR[b];
        part = fma((v.x * v.x + v.y * v.y) * (la * la), lb * lb, part);
      }
      acc = fma((double)i, part, acc);
    }
  }
  const double tot = block_sum(acc, sh);
  if (threadIdx.x == 0) out[s] = tot;
}

// S_k = - sum lambda^2 ln lambda^2 ; one CTA per bond
__global__ void __launch_bounds__(RD_THREADS) entropy_kernel(DevState S, double* out) {
  __shared__ double sh[RD_THREADS];
  const int k = blockIdx.x, NC = S.NC;
  int D = 0;
  for (int c = 0; c < NC; ++c) D += S.nb[(long long)k * NC + c];
  double acc = 0.0;
  for (int j = threadIdx.x; j < D; j += RD_THREADS) {
    const double l = S.lam[(long long)k * S.chi + j];
    const double p = l * l;
    if (p > 0.0) acc -= p * log(p);
  }
  const double tot = block_sum(acc, sh);
  if (threadIdx.x == 0) out[k] = tot;
}

// block offsets of one site from the two bond tables (after an import)
__global__ void gamoff_kernel(DevState S, int s) {
  if (threadIdx.x != 0 || blockIdx.x != 0) return;
  const int NC = S.NC, d = S.d;
  long long off = 0;
  for (int cl = 0; cl < NC; ++cl)
    for (int i = 0; i < d; ++i) {
      S.gamoff[((long long)s * NC + cl) * d + i] = off;
      if (cl - i >= 0) off += (long long)S.nb[(long long)s * NC + cl] * S.nb[(long long)(s + 1) * NC + cl - i];
    }
}

// |occ>: every bond one sector of multiplicity 1 (SURVEY §8(c) State)
__global__ void product_state_kernel(DevState S, const int* occ) {
  if (blockIdx.x != 0) return;
  const int NC = S.NC, M = S.M, d = S.d;
  for (long long i = threadIdx.x; i < (long long)(M + 1) * NC; i += blockDim.x) { S.nb[i] = 0; S.ob[i] = 0; }
  for (long long i = threadIdx.x; i < (long long)M * NC * d; i += blockDim.x) S.gamoff[i] = 0;
  __syncthreads();
  if (threadIdx.x == 0) {
    int c = S.N;
    for (int k = 0; k <= M; ++k) {
      S.nb[(long long)k * NC + c] = 1;
      for (int c2 = c + 1; c2 < NC; ++c2) S.ob[(long long)k * NC + c2] = 1;
      S.lam[(long long)k * S.chi] = 1.0;
      if (k < M) {
        S.gam[(long long)k * S.gcap] = make_double2(1.0, 0.0);  // the only block with non-zero area, offset 0
        c -= occ[k];
      }
    }
    S.scal[0] = 0.0; S.scal[1] = 0.0; S.scal[2] = 1.0; S.scal[3] = 1.0;
    S.err[0] = 0; S.err[1] = 0; S.err[2] = 0;
  }
  __syncthreads();
  for (int s = threadIdx.x; s < M; s += blockDim.x) {
    long long off = 0;
    for (int cl = 0; cl < NC; ++cl)
      for (int i = 0; i < d; ++i) {
        S.gamoff[((long long)s * NC + cl) * d + i] = off;
        if (cl - i >= 0) off += (long long)S.nb[(long long)s * NC + cl] * S.nb[(long long)(s + 1) * NC + cl - i];
      }
  }
}

void u1_launch_expect_n(const DevState& S, double* out_dev, const LaunchCfg& L) {
  L.prof->begin(U1_ST_READOUT, L.stream);
  expect_n_kernel<<<S.M, RD_THREADS, 0, L.stream>>>(S, out_dev);
  L.prof->end(L.stream);
  ++*L.launches;
}
void u1_launch_entropy(const DevState& S, double* out_dev, const LaunchCfg& L) {
  L.prof->begin(U1_ST_READOUT, L.stream);
  entropy_kernel<<<S.M + 1, RD_THREADS, 0, L.stream>>>(S, out_dev);
  L.prof->end(L.stream);
  ++*L.launches;
}
void u1_launch_product_state(const DevState& S, const int* occ_dev, const LaunchCfg& L) {
  product_state_kernel<<<1, 256, 0, L.stream>>>(S, occ_dev);
  ++*L.launches;
}
void u1_launch_gamoff(const DevState& S, int site, const LaunchCfg& L) {
  gamoff_kernel<<<1, 32, 0, L.stream>>>(S, site);
  ++*L.launches;
}
