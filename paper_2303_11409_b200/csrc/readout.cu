// readout.cu — step a6 (canonical-form readouts, SURVEY §8(c) "Readouts"; Eq.10/15 canonical form)
// and the small state-maintenance kernels (product state, block-offset rebuild after an import).
#include <algorithm>
#include <mutex>
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

// <n_s> = sum_{cl,cr} (cl - cr) sum_{a,b} lamL[cl]_a^2 |Gamma[cl,cr]_ab|^2 lamR[cr]_b^2   (canonical form, Eq.10/15)
// Memory-bound: every Gamma block with occupation >= 1 is read once.  The rows of all such blocks of a site form one
// virtual row space; slice j of K of it belongs to CTA (site, j) - K is chosen by the host so that all SMs are busy
// whatever M is - one warp per row, lanes along the row (coalesced 16-byte loads), shuffle reductions.  The K partial
// sums of a site are added in slice order by the last CTA of the site: the result does not depend on timing.
#define RD_UNR 8          // 16-byte loads in flight per thread
#define RD_MAXBLK 1024   // (cl, i) blocks of a site held in shared memory at a time (more are processed in batches)
__global__ void __launch_bounds__(RD_THREADS) expect_n_kernel(DevState S, int site0, int K, double* part, int* count, double* out) {
  __shared__ int s_pref[RD_MAXBLK + 1];        // virtual row prefix over the blocks of the batch
  __shared__ int s_cl[RD_MAXBLK];               // block -> cl * d + i
  __shared__ double s_red[RD_THREADS / 32];
  __shared__ int s_nblk, s_last;
  const int s = site0 + blockIdx.x / K, j = blockIdx.x % K, NC = S.NC, d = S.d;
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  const int* nbL = S.nb + (long long)s * NC;
  const int* nbR = S.nb + (long long)(s + 1) * NC;
  const cplx* gam = S.gam + (long long)s * S.gcap;
  const long long* goff = S.gamoff + (long long)s * NC * d;
  const double* lamL0 = S.lam + (long long)s * S.chi;
  const double* lamR0 = S.lam + (long long)(s + 1) * S.chi;
  const int* obL = S.ob + (long long)s * NC;
  const int* obR = S.ob + (long long)(s + 1) * NC;
  double acc = 0.0;   // this thread's sum
  for (int f0 = 0; f0 < NC * d; f0 += RD_MAXBLK) {   // batches of candidate (cl, i) pairs (one batch unless NC * d > 1024)
    __syncthreads();
    // rows of every candidate block (0: absent, or occupation 0, which contributes nothing), all threads; then one
    // thread compacts the list out of shared memory
    for (int f = f0 + tid; f < min(NC * d, f0 + RD_MAXBLK); f += RD_THREADS) {
      const int cl = f / d, i = f - cl * d;
      s_cl[f - f0] = (i == 0 || cl - i < 0 || nbR[cl - i] == 0) ? 0 : nbL[cl];
    }
    __syncthreads();
    if (tid == 0) {
      int nb = 0, run = 0;
      for (int f = f0; f < min(NC * d, f0 + RD_MAXBLK); ++f) {
        const int rows = s_cl[f - f0];
        if (rows == 0) continue;
        s_pref[nb] = run; s_cl[nb] = f; run += rows; ++nb;   // nb <= f - f0: the compacted list never overtakes the scan
      }
      s_pref[nb] = run; s_nblk = nb;
    }
    __syncthreads();
    const int nblk = s_nblk, rtot = s_pref[nblk];
    // rows [r0, r1) of the virtual row space belong to this slice.  Inside a block these rows are one contiguous array:
    // the CTA streams it flat (thread t takes elements t, t + 256, ...: fully coalesced whatever the row length is),
    // row and column of an element from its index by a single-precision reciprocal (exact below 2^24) with a +-1 fix-up
    const int r0 = (int)((long long)rtot * j / K), r1 = (int)((long long)rtot * (j + 1) / K);
    int bi = 0;
    while (bi < nblk && s_pref[bi + 1] <= r0) ++bi;
    for (; bi < nblk && s_pref[bi] < r1; ++bi) {
      const int f = s_cl[bi], cl = f / d, i = f - cl * d, cr = cl - i;
      const int ra = max(r0, s_pref[bi]) - s_pref[bi], rb = min(r1, s_pref[bi + 1]) - s_pref[bi];
      const int nr = nbR[cr];
      const cplx* blk = gam + goff[f] + (long long)ra * nr;
      const double* lamL = lamL0 + obL[cl] + ra;
      const double* lamR = lamR0 + obR[cr];
      const int ne = (rb - ra) * nr;              // <= chi^2 = 2^24
      const float inv = 1.0f / (float)nr;
      double p = 0.0;
      for (int e0 = tid; e0 < ne; e0 += RD_UNR * RD_THREADS) {
        cplx v[RD_UNR]; double w[RD_UNR];
#pragma unroll
        for (int x = 0; x < RD_UNR; ++x) {
          const int idx = e0 + x * RD_THREADS;
          const bool ok = idx < ne;
          v[x] = ok ? __ldcs(blk + idx) : make_double2(0.0, 0.0);
          int ar = __float2int_rz((float)idx * inv), br = idx - ar * nr;
          if (br >= nr) { br -= nr; ++ar; } else if (br < 0) { br += nr; --ar; }
          const double la = ok ? lamL[ar] : 0.0, lb = ok ? lamR[br] : 0.0;
          w[x] = (la * la) * (lb * lb);
        }
#pragma unroll
        for (int x = 0; x < RD_UNR; ++x) p = fma(fma(v[x].x, v[x].x, v[x].y * v[x].y), w[x], p);
      }
      acc = fma((double)i, p, acc);
    }
  }
  // deterministic sum over the CTA: lanes by shuffle, warps in order
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) acc += __shfl_xor_sync(0xffffffffu, acc, o);
  if (lane == 0) s_red[warp] = acc;
  __syncthreads();
  if (tid == 0) {
    double t = 0.0;
    for (int w = 0; w < RD_THREADS / 32; ++w) t += s_red[w];
    part[(long long)(s - site0) * K + j] = t;
    __threadfence();
    s_last = (atomicAdd(&count[s - site0], 1) == K - 1) ? 1 : 0;
  }
  __syncthreads();
  if (s_last && tid == 0) {   // the slices of the site, in slice order
    __threadfence();
    double t = 0.0;
    for (int jj = 0; jj < K; ++jj) t += __ldcg(&part[(long long)(s - site0) * K + jj]);
    out[s] = t;
    count[s - site0] = 0;     // ready for the next launch
  }
}

// S_k = - sum lambda^2 ln lambda^2 ; one CTA per bond
__global__ void __launch_bounds__(RD_THREADS) entropy_kernel(DevState S, int bond0, double* out) {
  __shared__ double sh[RD_THREADS];
  const int k = bond0 + blockIdx.x, NC = S.NC;
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

void u1_launch_expect_n(const DevState& S, int site0, int nsites, double* part, int* count, double* out_dev, const LaunchCfg& L) {
  // K slices per site so that the grid is one full wave of resident CTAs whatever the number of sites is
  static int occ = 0;
  if (occ == 0 && cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, expect_n_kernel, RD_THREADS, 0) != cudaSuccess) occ = 4;
  const int K = std::max(1, std::min(U1_RD_SLICES, (std::max(occ, 1) * L.sms) / nsites));
  L.prof->begin(U1_ST_READOUT, L.stream);
  expect_n_kernel<<<nsites * K, RD_THREADS, 0, L.stream>>>(S, site0, K, part, count, out_dev);
  L.prof->end(L.stream);
  ++*L.launches;
}
void u1_launch_entropy(const DevState& S, int bond0, int nbonds, double* out_dev, const LaunchCfg& L) {
  L.prof->begin(U1_ST_READOUT, L.stream);
  entropy_kernel<<<nbonds, RD_THREADS, 0, L.stream>>>(S, bond0, out_dev);
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

// ---- step a6 on library-owned static scratch: u1mps_expect_n_all_static (include/u1mps.h) --------------------------
// The same expect_n_kernel, with the slice partial sums and the per-site slice counters in a file-scope device array
// instead of the handle's arena, for callers that must not allocate (CUDA graph capture, serving loops): the call makes
// no cudaMalloc / cudaFree and no allocating library call, only a memset node and one kernel launch on the handle's stream.
// The array costs U1_RD_STATIC_BYTES (68 KiB) on every GPU that loads the library, until the process exits.  All handles
// and all calls share it: two calls that overlap on the GPU (different streams, no ordering) race on it.  The counters
// must start at zero, so every call clears the ones it uses first (the kernel also resets them when a site completes,
// but a call that was aborted half way would otherwise poison the next one); the partial sums are written before read.
#define U1_RD_STATIC_PART 8192                                                   // slice partial sums (doubles)
#define U1_RD_STATIC_BYTES (U1_RD_STATIC_PART * 8 + U1_RD_STATIC_SITES * 4)      // + one counter per site = 69 632 bytes
static __device__ __align__(256) unsigned char rd_static_scratch[U1_RD_STATIC_BYTES];

#define U1_RD_MAXDEV 64
// In host code `rd_static_scratch` is only the host-side shadow of the symbol, never a device address: the address
// comes from cudaGetSymbolAddress, once per device, with that device current.
static cudaError_t rd_static_address(unsigned char** out) {
  static std::mutex mu;
  static unsigned char* addr[U1_RD_MAXDEV] = {};
  int dev = -1;
  cudaError_t e = cudaGetDevice(&dev);
  if (e != cudaSuccess) return e;
  if (dev < 0 || dev >= U1_RD_MAXDEV) return cudaErrorInvalidDevice;
  std::lock_guard<std::mutex> lock(mu);
  if (!addr[dev]) {
    void* p = nullptr;
    e = cudaGetSymbolAddress(&p, rd_static_scratch);
    if (e != cudaSuccess) return e;
    addr[dev] = static_cast<unsigned char*>(p);
  }
  *out = addr[dev];
  return cudaSuccess;
}

// nsites <= U1_RD_STATIC_SITES is the caller's check (api.cu turns a larger chain into U1MPS_ETOOBIG); out_dev: DEVICE
// double[nsites], sites 0 .. nsites - 1.  Not timed by the stage profiler (its event pool may allocate).
cudaError_t u1_launch_expect_n_static(const DevState& S, int nsites, double* out_dev, const LaunchCfg& L) {
  if (nsites < 1 || nsites > U1_RD_STATIC_SITES) return cudaErrorInvalidValue;
  unsigned char* base = nullptr;
  cudaError_t e = rd_static_address(&base);
  if (e != cudaSuccess) return e;
  double* part = reinterpret_cast<double*>(base);
  int* count = reinterpret_cast<int*>(base + (size_t)U1_RD_STATIC_PART * 8);
  static int occ = 0;
  if (occ == 0 && cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, expect_n_kernel, RD_THREADS, 0) != cudaSuccess) occ = 4;
  int K = std::max(1, std::min(U1_RD_SLICES, (std::max(occ, 1) * L.sms) / nsites));   // as u1_launch_expect_n ...
  K = std::min(K, U1_RD_STATIC_PART / nsites);                                         // ... within the static array (>= 8)
  e = cudaMemsetAsync(count, 0, (size_t)nsites * sizeof(int), L.stream);
  if (e != cudaSuccess) return e;
  expect_n_kernel<<<nsites * K, RD_THREADS, 0, L.stream>>>(S, 0, K, part, count, out_dev);
  ++*L.launches;
  return cudaGetLastError();
}
