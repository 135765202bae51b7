// rt_device.cuh -- device-side building blocks shared by the sm_100a kernels of this library.
// (Nothing here is shared with oracle/: the oracle has its own Philox, draw and propensity.)
//
// All fp64 arithmetic that decides a result uses the rounding-explicit intrinsics
// (__dmul_rn / __dadd_rn / __dsub_rn / __ddiv_rn), which nvcc never contracts into FMAs, so
// every operation is one IEEE round-to-nearest step in the order DESIGN.md fixes.
#pragma once
#include <cstdint>
#include <cuda_runtime.h>

namespace rt {

typedef unsigned long long u64;

// Device copy of the network (rt_network of include/rt.h) plus the dependency lists.
struct NetDev {
  int32_t N, M;
  int32_t M_pad;                 // M rounded up to even; entry M (if any) has a = 0, T = P = 0
  const uint32_t *react_ptr;     // [M+1]
  const int32_t *react_species;  // [nnz_r]
  const int32_t *react_sigma;    // [nnz_r]
  const uint32_t *stoich_ptr;    // [M+1]
  const int32_t *stoich_species; // [nnz_v]
  const int32_t *stoich_v;       // [nnz_v]
  const double *rate;            // [M]
  // Dependency graph, stored two-hop and dense so that a walk is three
  // dependent loads: stoich row of mu -> species record -> dependency entries.
  const int32_t *srow;           // [M][4][4] ELL copy of the stoich row of k, 64 B: per changed species
                                 //        (j, v, lo, hi): [lo, hi) = its entries in dep[]; hubs store
                                 //        (j, v, row of big_off, 0xffffffff); unused slot j = -1;
                                 //        srow[k][0].j = -2: more than 4 entries, walk the CSR row
  const uint32_t *sp_rec;        // [N][2] (lo, hi): entries of species j in dep[]
  const int32_t *sp_big;         // [N]    row of big_off for hub species (degree > big_deg), else -1
  const uint32_t *big_off;       // [n_big][n_blk+1] hub species: first entry with k >= b << blk_shift
  const int32_t *dep;            // [nnz_r] 32-byte entries, sorted by k within a species:
                                 //        int32 k, j1, j2 (or -1), sigma1 | sigma2 << 8 | general << 16;
                                 //        double c_k; 8 bytes padding.  (j1, j2) = first two reactants
  int32_t n_blk, blk_shift, big_deg;
  long long xmax;                // count bound (2^31-1, or 2^21-1 if some sigma = 3)
};

// ------------------------------------------------------------------ Philox4x32-10
// Salmon et al., SC'11.  Returns output words 0 and 1 (the two the draw uses).
__device__ __forceinline__ void philox4x32_10(uint32_t c0, uint32_t c1, uint32_t c2, uint32_t c3,
                                              uint32_t k0, uint32_t k1,
                                              uint32_t &o0, uint32_t &o1) {
#pragma unroll
  for (int i = 0; i < 10; ++i) {
    const uint32_t hi0 = __umulhi(0xD2511F53u, c0), lo0 = 0xD2511F53u * c0;
    const uint32_t hi1 = __umulhi(0xCD9E8D57u, c2), lo1 = 0xCD9E8D57u * c2;
    c0 = hi1 ^ c1 ^ k0;
    c1 = lo1;
    c2 = hi0 ^ c3 ^ k1;
    c3 = lo0;
    k0 += 0x9E3779B9u;
    k1 += 0xBB67AE85u;
  }
  o0 = c0;
  o1 = c1;
}

// n-th unit-exponential increment of channel k (Eq.23: Delta T = ln(1/r)).
// key = (lo32 seed, hi32 seed), counter = (k, n, lo32 traj, hi32 traj);
// r = (u53 + 1) * 2^-53 in (0, 1].
// (not inlined: Philox + log is ~4 KB of code, and the per-firing loop has to stay in the
// instruction cache)
__device__ __noinline__ double exp_draw(u64 seed, u64 traj, uint32_t k, uint32_t n) {
  uint32_t w0, w1;
  philox4x32_10(k, n, (uint32_t)traj, (uint32_t)(traj >> 32), (uint32_t)seed,
                (uint32_t)(seed >> 32), w0, w1);
  const u64 u53 = (((u64)w1 << 32) | (u64)w0) >> 11;
  const double r = __dmul_rn(__ull2double_rn(u53 + 1ull), 0x1.0p-53);
  return -log(r);
}

// C(x, sigma), exact integer (Eq.2; reading G2).
__device__ __forceinline__ long long binom(long long x, int sigma) {
  if (sigma == 1) return x;
  const long long h = x * (x - 1) / 2;
  if (sigma == 2) return h;
  return h * (x - 2) / 3;
}

// The bundle kernel keeps ONE copy of X per trajectory in global memory (L2-resident), each
// word = (version << 31) | count: version = index of the firing that last changed the species
// (1-based, 33 bits), count < 2^31.  Every CTA applies every firing's update itself with
// atomicMax (red.max.u64): all CTAs write the same word, and a delayed write of an older firing
// can never replace a newer one, so no fence sits between a firing and the next.
constexpr int kXCountBits = 31;
constexpr u64 kXCountMask = (1ull << kXCountBits) - 1ull;
constexpr u64 kXMaxVersion = (1ull << (64 - kXCountBits)) - 2ull;
__device__ __forceinline__ long long x_count(u64 w) { return (long long)(w & kXCountMask); }
__device__ __forceinline__ u64 x_version(u64 w) { return w >> kXCountBits; }
__device__ __forceinline__ u64 x_pack(u64 version, long long count) {
  return (version << kXCountBits) | (u64)count;
}
__device__ __forceinline__ long long x_load(const u64 *Xv, int j) { return x_count(__ldcg(Xv + j)); }

// a_k = c_k * prod_j C(X_j, sigma_jk): one rounded multiply per reactant, CSR order.
// X is read with ld.global.cg (L2): other CTAs write it too.  Not inlined (code size); takes the
// arrays rather than the NetDev so that no copy of the kernel parameters is forced into local memory.
__device__ __noinline__ double propensity_csr(double c, const uint32_t *react_ptr,
                                              const int32_t *react_species, const int32_t *react_sigma,
                                              const u64 *Xv, int k) {
  double a = c;
  const uint32_t e1 = __ldg(react_ptr + k + 1);
  for (uint32_t e = __ldg(react_ptr + k); e < e1; ++e) {
    const long long x = x_load(Xv, __ldg(react_species + e));
    a = __dmul_rn(a, __ll2double_rn(binom(x, __ldg(react_sigma + e))));
  }
  return a;
}
__device__ __forceinline__ double propensity(const NetDev &net, const u64 *Xv, int k) {
  return propensity_csr(__ldg(net.rate + k), net.react_ptr, net.react_species, net.react_sigma, Xv, k);
}

// ------------------------------------------------------------------ lexicographic argmin
struct Cand {
  double dt;
  int k;
};
__device__ __forceinline__ bool cand_less(double dt, int k, const Cand &b) {
  return dt < b.dt || (dt == b.dt && k < b.k);
}
// Warp-wide lexicographic min of (dt, k), result in every lane.  dt >= 0 (or +inf), never NaN, so
// its bit pattern orders like an unsigned integer: three REDUX.MIN steps (high word, low word
// among the lanes that tie on the high word, k among the lanes that tie on both) replace five
// rounds of 64-bit shuffles.
__device__ __forceinline__ Cand warp_lexmin(Cand c) {
  const unsigned hi = (unsigned)__double2hiint(c.dt), lo = (unsigned)__double2loint(c.dt);
  const unsigned h = __reduce_min_sync(0xffffffffu, hi);
  const unsigned l = __reduce_min_sync(0xffffffffu, hi == h ? lo : 0xffffffffu);
  const unsigned k = __reduce_min_sync(0xffffffffu, (hi == h && lo == l) ? (unsigned)c.k : 0xffffffffu);
  Cand r;
  r.dt = __hiloint2double((int)h, (int)l);
  r.k = (int)k;
  return r;
}

// Waiting time of one channel (Eq.24 with constant a_k; readings G4, G7): a = 0 gives +inf.
__device__ __forceinline__ double waiting_time(double P, double T, double a) {
  if (!(a > 0.0)) return __longlong_as_double(0x7ff0000000000000ll);
  double r = __dsub_rn(P, T);
  r = r < 0.0 ? 0.0 : r;
  return __ddiv_rn(r, a);
}

// ------------------------------------------------------------------ memory-model helpers
__device__ __forceinline__ void st_release_u32(uint32_t *p, uint32_t v) {
  asm volatile("st.release.gpu.global.u32 [%0], %1;" ::"l"(p), "r"(v) : "memory");
}
__device__ __forceinline__ uint32_t ld_acquire_u32(const uint32_t *p) {
  uint32_t v;
  asm volatile("ld.acquire.gpu.global.u32 %0, [%1];" : "=r"(v) : "l"(p) : "memory");
  return v;
}
__device__ __forceinline__ void prefetch_l2(const void *p) {
  asm volatile("prefetch.global.L2 [%0];" ::"l"(p));
}
__device__ __forceinline__ void st_relaxed_v2(u64 *p, u64 a, u64 b) {
  asm volatile("st.relaxed.gpu.global.v2.u64 [%0], {%1, %2};" ::"l"(p), "l"(a), "l"(b) : "memory");
}
__device__ __forceinline__ void ld_relaxed_v2(const u64 *p, u64 &a, u64 &b) {
  asm volatile("ld.relaxed.gpu.global.v2.u64 {%0, %1}, [%2];" : "=l"(a), "=l"(b) : "l"(p) : "memory");
}


// ------------------------------------------------------------------ thread-block clusters (DSMEM)
// A bundle of at most kMaxClusterCtas CTAs is launched as ONE thread-block cluster: its per-firing
// exchange then never leaves the SMs (remote shared-memory stores that signal the receiver's
// mbarrier), instead of a store -> load hand-over through L2.
constexpr int kMaxClusterCtas = 16;
__device__ __forceinline__ uint32_t smem_addr(const void *p) { return (uint32_t)__cvta_generic_to_shared(p); }
// shared::cluster address of this CTA's shared-memory address `addr` in the CTA of rank `rank`
__device__ __forceinline__ uint32_t mapa_u32(uint32_t addr, uint32_t rank) {
  uint32_t r;
  asm volatile("mapa.shared::cluster.u32 %0, %1, %2;" : "=r"(r) : "r"(addr), "r"(rank));
  return r;
}
__device__ __forceinline__ void mbar_init(uint32_t bar, uint32_t count) {
  asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(bar), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_fence_init() {
  asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
}
// one arrival that also announces `bytes` of st.async traffic for the current phase
__device__ __forceinline__ void mbar_arrive_expect_tx(uint32_t bar, uint32_t bytes) {
  asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(bar), "r"(bytes) : "memory");
}
__device__ __forceinline__ bool mbar_try_wait(uint32_t bar, uint32_t parity) {
  uint32_t ok;
  asm volatile("{\n .reg .pred p;\n mbarrier.try_wait.parity.acquire.cluster.shared::cta.b64 p, [%1], %2;\n"
               " selp.u32 %0, 1, 0, p;\n}" : "=r"(ok) : "r"(bar), "r"(parity) : "memory");
  return ok != 0;
}
// 16-byte store into a peer CTA's shared memory; completes 16 bytes on the peer's mbarrier `rbar`
__device__ __forceinline__ void st_async_v2(uint32_t raddr, u64 a, u64 b, uint32_t rbar) {
  asm volatile("st.async.weak.shared::cluster.mbarrier::complete_tx::bytes.v2.b64 [%0], {%1, %2}, [%3];"
               ::"r"(raddr), "l"(a), "l"(b), "r"(rbar) : "memory");
}
__device__ __forceinline__ void cluster_barrier() {     // every thread of every CTA of the cluster
  asm volatile("barrier.cluster.arrive.release.aligned;\n barrier.cluster.wait.acquire.aligned;" ::: "memory");
}

}  // namespace rt
