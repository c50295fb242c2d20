// common.cuh — device-side data layout shared by the kernels of libu1mps.so (product path only;
// nothing here is shared with oracle/).  See DESIGN.md §"Data layout in HBM".
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

typedef double2 cplx;  // complex128, interleaved (x = re, y = im), 16-byte aligned

#define U1_TILE 32         // a2 / a5 tile edge
#define U1_MAXSWEEP 30     // Jacobi (outer) sweep limit
#define U1_PB 16           // columns per Jacobi panel: a pair item orthogonalises 2*U1_PB = 32 columns
#define U1_ERR_WORKSPACE 1 // device error flag: plan does not fit the workspace
#define U1_ERR_SCHED 2     // device error flag: an a3 work-queue dependency did not resolve (internal error)
#define U1_RD_SLICES 1024   // a6: at most this many CTAs share one site
#define U1_RD_STATIC_SITES 1024   // a6 on static scratch: longest chain (= U1MPS_STATIC_SITES_MAX of include/u1mps.h)
#define U1_SCHED 264       // entries of Plan::sched
#define U1_SVD_THREADS 128 // 4 warps per pair item, 6 CTAs per SM
#define U1MPS_SORT_MAX 4096 // largest sector the in-smem bitonic sort takes (= U1MPS_CHI_MAX)

// Persistent MPS state (all device pointers into the caller's arena).
struct DevState {
  int M, d, N, NC, chi;  // NC = N + 1 charge values 0..N
  int* nb;               // [(M+1)*NC]  n_k(c): multiplicity of charge c on bond k (0 = absent)
  int* ob;               // [(M+1)*NC]  exclusive scan of nb over c: offset of sector c in lambda^[k]
  double* lam;           // [(M+1)*chi] lambda^[k], sectors ascending c, descending inside
  cplx* gam;             // [M*gcap]    Gamma^[s] blocks, each row-major n_s(cl) x n_{s+1}(cr), tightly packed
  long long gcap;        // chi*chi elements per site
  long long* gamoff;     // [M*NC*d]    offset of block (cl, i = cl-cr) inside site s (scan over (cl,i))
  double* scal;          // [0] log-norm, [1] discarded weight (total), [2] last w_kept, [3] last w_all
  int* err;              // [0] sticky device error flag, [1] sweeps used (max), [2] non-converged blocks
};

// Per-launch plan for a batch ("chunk") of G disjoint gates.  Entry e = g*NC + c is the candidate
// centre charge c of gate g (rows == 0 means "not a candidate").
struct Plan {
  int* site;         // [G] left site of gate g
  cplx* U;           // [G*d^4] gate matrices
  int* rows;         // [G*NC] rows(c) = sum_i n_L(c+i)
  int* cols;         // [G*NC] cols(c) = sum_j n_R(c-j)
  long long* goff;   // [G*NC+1] offset of the stacked (m+n) x n column-major Jacobi matrix of entry e
  int* svoff;        // [G*NC+1] exclusive scan of n = min(rows, cols): offset in the sigma pool
  int* t2pref;       // [G*NC*d*d+1] a2 tile prefix over (e, i, j)
  int* t5pref;       // [G*NC*2+1] a5 tile prefix over (e, part)  part 0 = V, 1 = W
  int* blk;          // [G*NC] compact list of entries with n > 0
  int* pitem_e;      // [cap] Jacobi panel-pair items: entry e
  int* pitem_k;      // [cap] ... pair slot k of the round-robin tournament
  int* tmpa;         // [G*NC+1] scratch: pair-item offset per entry
  int* cnt;          // [8] 0: #blk, 1: #pair items, 3: max panels (even), 4: a2 tiles, 5: a5 tiles, 7: a4 CTA counter
  int* sched;        // [U1_SCHED] a3 scheduling state of one launch: work counters, tickets, CTA ranks per SM (svd.cu)
  int* flags;        // [3*G*NC] a3 per entry: round after the last counting rotation, round found finished, items completed
  long long* trace;  // [4*U1_MAXSWEEP] a3 trace of the last launch: per sweep end time (globaltimer ns), rotated items, inner sweeps, active sectors
  int* keep;         // [G*NC] kept singular values per entry (a4)
  int* perm;         // [pool] sorted position -> column index
  double* sv;        // [pool] unsorted column norms
  double* svs;       // [pool] sorted descending
  double* gate_w;    // [2*G] per gate: kept weight, total weight (a4)
  cplx* W;           // workspace for the stacked Jacobi matrices
  long long wcap;    // capacity of W in elements
  int poolcap;       // capacity of sv / svs / perm
  int itemcap;       // capacity of the item lists
};

__host__ __device__ inline int u1_ceil_div(int a, int b) { return (a + b - 1) / b; }

#ifdef __CUDACC__
// D(8x8) += A(8x4, row) * B(4x8, col), FP64 tensor tile (SASS: DMMA.8x8x4).
// Fragments: a = A[lane>>2][lane&3], b = B[lane&3][lane>>2], c0/c1 = C[lane>>2][2*(lane&3) + 0/1].
__device__ __forceinline__ void dmma(double& c0, double& c1, double a, double b) {
  asm("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};\n" : "+d"(c0), "+d"(c1) : "d"(a), "d"(b));
}

// Exclusive scan of f(0..L-1) into out[0..L] (out[L] = total) by one CTA of NT threads; sh: NT entries of shared memory.
template <typename T, int NT, typename F>
__device__ void u1_block_excl_scan(F f, T* out, int L, T* sh) {
  const int t = threadIdx.x;
  const int per = (L + NT - 1) / NT;
  const int lo = min(L, t * per), hi = min(L, lo + per);
  T sum = 0;
  for (int i = lo; i < hi; ++i) sum += f(i);
  sh[t] = sum;
  __syncthreads();
  for (int off = 1; off < NT; off <<= 1) {  // Hillis-Steele inclusive scan
    T v = (t >= off) ? sh[t - off] : (T)0;
    __syncthreads();
    sh[t] += v;
    __syncthreads();
  }
  T run = sh[t] - sum;
  for (int i = lo; i < hi; ++i) { T v = f(i); out[i] = run; run += v; }
  if (t == NT - 1) out[L] = sh[t];
  __syncthreads();
}
#endif

// Optional per-kernel timing (u1mps_profile_*): CUDA events recorded on the handle's stream around
// every launch of a stage; summed when read.  Host side only.
enum { U1_ST_PLAN = 0, U1_ST_CONTRACT, U1_ST_IDENTITY, U1_ST_SVD, U1_ST_SORT, U1_ST_SELECT, U1_ST_SCATTER, U1_ST_READOUT, U1_NSTAGE };
#include <vector>
struct Prof {
  bool on = false;
  std::vector<cudaEvent_t> pool;     // begin/end pairs, reused
  std::vector<int> stage;            // stage of pair i
  size_t used = 0;                   // pairs in flight
  void begin(int st, cudaStream_t s) {
    if (!on) return;
    if (used == stage.size()) {
      cudaEvent_t a, b;
      if (cudaEventCreate(&a) != cudaSuccess || cudaEventCreate(&b) != cudaSuccess) { on = false; return; }
      pool.push_back(a); pool.push_back(b); stage.push_back(st);
    }
    stage[used] = st;
    cudaEventRecord(pool[2 * used], s);
  }
  void end(cudaStream_t s) {
    if (!on) return;
    cudaEventRecord(pool[2 * used + 1], s);
    ++used;
  }
  void destroy() { for (cudaEvent_t e : pool) cudaEventDestroy(e); pool.clear(); stage.clear(); used = 0; }
};

// Host-side launchers (one per kernel file).  `stream` is the handle's stream.
struct LaunchCfg { int sms; int svd_grid; int svd_smem; cudaStream_t stream; long long* launches; Prof* prof; };

void u1_launch_plan(const DevState& S, const Plan& P, int G, const LaunchCfg& L);
void u1_launch_contract(const DevState& S, const Plan& P, int G, const LaunchCfg& L);
cudaError_t u1_launch_svd(const DevState& S, const Plan& P, int G, const LaunchCfg& L);
void u1_launch_select_scatter(const DevState& S, const Plan& P, int G, int chi, double cutoff, const LaunchCfg& L);
void u1_launch_expect_n(const DevState& S, int site0, int nsites, double* part, int* count, double* out_dev, const LaunchCfg& L);
cudaError_t u1_launch_expect_n_static(const DevState& S, int nsites, double* out_dev, const LaunchCfg& L);   // no allocation
void u1_launch_entropy(const DevState& S, int bond0, int nbonds, double* out_dev, const LaunchCfg& L);
void u1_launch_product_state(const DevState& S, const int* occ_dev, const LaunchCfg& L);
void u1_launch_gamoff(const DevState& S, int site, const LaunchCfg& L);
cudaError_t u1_svd_configure(int* grid, int* smem_bytes, int sms);
size_t u1_env_scratch_bytes(int M, int NC, int d, const std::vector<int>& nb, const std::vector<long long>& gused);
size_t u1_env_nn_scratch_bytes(int M, int NC, int d, const std::vector<int>& nb, const std::vector<long long>& gused);
cudaError_t u1_env_expect_nn(const DevState& S, const std::vector<int>& nb, const std::vector<long long>& gamoff,
                             const std::vector<long long>& gused, int j, int k, void* scratch, double* out_dev, const LaunchCfg& L);
size_t u1_env_sample_scratch_bytes(int M, int NC, int d, const std::vector<int>& nb, const std::vector<long long>& gused, int B);
cudaError_t u1_env_sample_fock(const DevState& S, const std::vector<int>& nb, const std::vector<long long>& gamoff,
                               const std::vector<long long>& gused, int B, const double* u_host, int* pat_host, double* logp_host,
                               void* scratch, const LaunchCfg& L);
cudaError_t u1_env_expect_n(const DevState& S, const std::vector<int>& nb, const std::vector<long long>& gamoff,
                            const std::vector<long long>& gused, void* scratch, double* out_dev, const LaunchCfg& L);
