// plan.cu — step a1: sector enumeration and offsets ("a subset of bonds ... that satisfy
// the conditions on the three charges"; L121: 0 <= c^[k] <= N; Eq.16's deltas bound the occupations
// by d-1).  Integer only, one CTA, no host round trip: everything later kernels need to find their
// work (Theta offsets, tile lists, Jacobi item lists) is produced here from the three bond tables.
#include "common.cuh"

#define PLAN_THREADS 1024
#define U1_MAXPANELS (U1MPS_SORT_MAX / U1_PB)   // panels of the largest sector (n <= chi <= 4096)

__global__ void __launch_bounds__(PLAN_THREADS) plan_kernel(DevState S, Plan P, int G) {
  __shared__ long long shl[PLAN_THREADS];
  __shared__ int shi[PLAN_THREADS];
  __shared__ int shmax, sh_over;
  __shared__ int cls_count[U1_MAXPANELS + 1], cls_fill[U1_MAXPANELS + 1], cls_base[U1_MAXPANELS + 1];
  const int NC = S.NC, d = S.d, E = G * NC, t = threadIdx.x;
  if (t == 0) { shmax = 0; sh_over = 0; }
  // (i)-(iii) rows(c), cols(c) of every candidate centre charge
  for (int e = t; e < E; e += PLAN_THREADS) {
    const int g = e / NC, c = e % NC, s = P.site[g];
    const int* nL = S.nb + (long long)s * NC;
    const int* nR = S.nb + (long long)(s + 2) * NC;
    int r = 0, q = 0;
    for (int i = 0; i < d; ++i) {
      if (c + i <= S.N) r += nL[c + i];
      if (c - i >= 0) q += nR[c - i];
    }
    if (r == 0 || q == 0) r = q = 0;
    P.rows[e] = r;
    P.cols[e] = q;
    P.keep[e] = 0;
  }
  __syncthreads();
  // Theta / Jacobi workspace offsets: stacked (m+n) x n column-major, m = max(rows, cols), n = min
  u1_block_excl_scan<long long, PLAN_THREADS>(
      [&](int e) { long long r = P.rows[e], q = P.cols[e]; long long m = max(r, q), n = min(r, q); return (m + n) * n; },
      P.goff, E, shl);
  if (t == 0 && P.goff[E] > P.wcap) sh_over = 1;
  u1_block_excl_scan<int, PLAN_THREADS>([&](int e) { return min(P.rows[e], P.cols[e]); }, P.svoff, E, shi);
  if (t == 0 && P.svoff[E] > P.poolcap) sh_over = 1;
  // (iv) a2 tile list over (e, i, j): block (c_l = c+i, c_r = c-j) of Theta(c)
  const int dd = d * d;
  u1_block_excl_scan<int, PLAN_THREADS>(
      [&](int f) {
        const int e = f / dd, i = (f / d) % d, j = f % d;
        if (P.rows[e] == 0) return 0;
        const int g = e / NC, c = e % NC, s = P.site[g];
        if (c + i > S.N || c - j < 0) return 0;
        const int nl = S.nb[(long long)s * NC + c + i], nr = S.nb[(long long)(s + 2) * NC + c - j];
        return u1_ceil_div(nl, U1_TILE) * u1_ceil_div(nr, U1_TILE);
      },
      P.t2pref, E * dd, shi);
  // a5 tile list over (e, part): V rows x n, W n x cols
  u1_block_excl_scan<int, PLAN_THREADS>(
      [&](int f) {
        const int e = f >> 1;
        const int r = P.rows[e], q = P.cols[e], n = min(r, q);
        if (n == 0) return 0;
        return (f & 1) ? u1_ceil_div(n, U1_TILE) * u1_ceil_div(q, U1_TILE) : u1_ceil_div(r, U1_TILE) * u1_ceil_div(n, U1_TILE);
      },
      P.t5pref, E * 2, shi);
  // Jacobi block list and item lists
  auto panels = [&](int e) {  // column panels of U1_PB columns of the Jacobi matrix of entry e
    const int n = min(P.rows[e], P.cols[e]);
    return u1_ceil_div(n, U1_PB);
  };
  u1_block_excl_scan<int, PLAN_THREADS>([&](int e) { return min(P.rows[e], P.cols[e]) > 0 ? 1 : 0; }, P.tmpa, E, shi);
  for (int e = t; e < E; e += PLAN_THREADS)
    if (min(P.rows[e], P.cols[e]) > 0) P.blk[P.tmpa[e]] = e;
  if (t == 0) P.cnt[0] = P.tmpa[E];
  __syncthreads();
  // pair items: (p+1)/2 panel pairs per round of the round-robin tournament; a single panel is one item.
  // Items are listed by descending panel count (longest first): the a3 work queue hands them out in this order,
  // so that the stragglers of a round are its cheapest items.
  for (int i = t; i <= U1_MAXPANELS; i += PLAN_THREADS) { cls_count[i] = 0; cls_fill[i] = 0; }
  __syncthreads();
  for (int e = t; e < E; e += PLAN_THREADS) {
    const int p = panels(e);
    if (p > 0) atomicAdd(&cls_count[min(p, U1_MAXPANELS)], (p + 1) / 2);
  }
  __syncthreads();
  if (t == 0) {
    int run = 0;
    for (int key = U1_MAXPANELS; key >= 1; --key) { cls_base[key] = run; run += cls_count[key]; }
    cls_base[0] = run;  // total
    P.cnt[1] = run;
    P.cnt[4] = P.t2pref[E * dd];
    P.cnt[5] = P.t5pref[E * 2];
    if (run > P.itemcap) sh_over = 1;
  }
  __syncthreads();
  const bool ok = cls_base[0] <= P.itemcap;
  int mymax = 0;
  for (int e = t; e < E; e += PLAN_THREADS) {
    const int p = panels(e);
    if (p == 0 || !ok) continue;
    mymax = max(mymax, p);
    const int np = (p + 1) / 2, key = min(p, U1_MAXPANELS);
    const int off = cls_base[key] + atomicAdd(&cls_fill[key], np);
    for (int k = 0; k < np; ++k) { P.pitem_e[off + k] = e; P.pitem_k[off + k] = k; }
  }
  atomicMax(&shmax, mymax);
  for (int i = t; i < 3 * E; i += PLAN_THREADS) P.flags[i] = (i >= E && i < 2 * E) ? 0x7fffffff : 0;   // a3: last_rot[E], done_at[E], done_cnt[E]
  for (int i = t; i < 4 * U1_MAXSWEEP + 1; i += PLAN_THREADS) P.trace[i] = 0;
  for (int i = t; i < U1_SCHED; i += PLAN_THREADS) P.sched[i] = 0;
  __syncthreads();
  if (t == 0) {
    P.cnt[3] = shmax;
    // the plan does not fit the arena: report it, and hand every later kernel of the launch an EMPTY work list, so that
    // nothing is written through the oversize offsets
    if (sh_over) { atomicExch(S.err, U1_ERR_WORKSPACE); P.cnt[0] = 0; P.cnt[1] = 0; P.cnt[4] = 0; P.cnt[5] = 0; }
  }
}

void u1_launch_plan(const DevState& S, const Plan& P, int G, const LaunchCfg& L) {
  L.prof->begin(U1_ST_PLAN, L.stream);
  plan_kernel<<<1, PLAN_THREADS, 0, L.stream>>>(S, P, G);
  L.prof->end(L.stream);
  ++*L.launches;
}
