// exchange_floor.cu -- micro-benchmark behind the exchange design of rt_bundle.cuh (DESIGN.md 6.1,
// profiles/r2_exchange_floor.md).  Standalone: nvcc -O3 -gencode arch=compute_100a,code=sm_100a
// -o exchange_floor exchange_floor.cu && ./exchange_floor.  Not part of the library.
//
// It measures the per-round floor of an all-gather of one 16-byte (value, tag) word per CTA when
// NOTHING else is done between rounds -- i.e. the latency one firing pays for its argmin exchange
// (the bundle-level reduction) however fast the pass is:
//   l2      S CTAs post to slots in global memory (L2), each CTA polls all S slots
//           (st.relaxed.gpu / ld.relaxed.gpu, slot stride SLOT_STRIDE words, double-buffered by round parity;
//           a lane's loads are all in flight together, as in rt_bundle.cuh)
//   l2push  each CTA writes its word into a private row of every reader (S x S slots), so that a
//           polled line has ONE reader and is written by one CTA per slot
//   l2near  every slot exists in 4 copies 8 MiB apart; a CTA polls the copy it reads fastest
//           (l2copies: the same 4 stores, but everybody polls copy 0)
//   l2die   148 CTAs in two groups by SM id half (l2parity: by SM id parity, a control), each group
//           gathering on its own slots
//   dsmem   the C CTAs of one thread-block cluster post into every peer's shared memory with
//           st.async (remote store + complete_tx on the peer's mbarrier), each waits on its own
//           mbarrier: no global memory on the path
//   hybrid  dsmem inside clusters of C, then the cluster leaders post to L2 and every CTA polls
//           the n_clusters slots
//   hyblead dsmem inside clusters, only the leaders post and poll in L2, then each leader sends
//           the result to its peers with st.async
//   hybpush dsmem inside clusters, leaders write the cluster's word into a private row of every CTA
// Each round's posted value depends on the previous round's result, as in the real kernel.
#include <cstdio>
#include <cstdlib>
#include <cstdint>
#include <vector>
#include <cuda_runtime.h>
#include <cooperative_groups.h>

typedef unsigned long long u64;
#ifndef SLOT_STRIDE
#define SLOT_STRIDE 128
#endif
constexpr int kSlotStride = SLOT_STRIDE;   // u64 words between slots: 1 KiB as in rt_bundle.cuh (-DSLOT_STRIDE=32: 256 B)

#define CK(x) do { cudaError_t e_ = (x); if (e_ != cudaSuccess) { \
  printf("CUDA error %s at %s:%d\n", cudaGetErrorString(e_), __FILE__, __LINE__); exit(1); } } while (0)

__device__ __forceinline__ void st_relaxed_v2(u64 *p, u64 a, u64 b) {
  asm volatile("st.relaxed.gpu.global.v2.u64 [%0], {%1, %2};" ::"l"(p), "l"(a), "l"(b) : "memory");
}
__device__ __forceinline__ void ld_relaxed_v2(const u64 *p, u64 &a, u64 &b) {
  asm volatile("ld.relaxed.gpu.global.v2.u64 {%0, %1}, [%2];" : "=l"(a), "=l"(b) : "l"(p) : "memory");
}
__device__ __forceinline__ uint32_t smem_addr(const void *p) { return (uint32_t)__cvta_generic_to_shared(p); }
__device__ __forceinline__ uint32_t mapa(uint32_t addr, uint32_t rank) {
  uint32_t r;
  asm volatile("mapa.shared::cluster.u32 %0, %1, %2;" : "=r"(r) : "r"(addr), "r"(rank));
  return r;
}
__device__ __forceinline__ void mbar_init(uint32_t bar, uint32_t count) {
  asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(bar), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_expect_tx(uint32_t bar, uint32_t bytes) {
  asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(bar), "r"(bytes) : "memory");
}
__device__ __forceinline__ bool mbar_try_wait(uint32_t bar, uint32_t parity) {
  uint32_t ok;
  asm volatile("{\n .reg .pred p;\n mbarrier.try_wait.parity.acquire.cluster.shared::cta.b64 p, [%1], %2;\n"
               " selp.u32 %0, 1, 0, p;\n}" : "=r"(ok) : "r"(bar), "r"(parity) : "memory");
  return ok != 0;
}
__device__ __forceinline__ void st_async_v2(uint32_t raddr, u64 a, u64 b, uint32_t rbar) {
  asm volatile("st.async.weak.shared::cluster.mbarrier::complete_tx::bytes.v2.b64 [%0], {%1, %2}, [%3];"
               ::"r"(raddr), "l"(a), "l"(b), "r"(rbar) : "memory");
}
__device__ __forceinline__ void cluster_sync_all() {
  asm volatile("barrier.cluster.arrive.release.aligned;\n barrier.cluster.wait.acquire.aligned;" ::: "memory");
}
__device__ __forceinline__ uint32_t cluster_rank() {
  uint32_t r; asm volatile("mov.u32 %0, %%cluster_ctarank;" : "=r"(r)); return r;
}

// Lane l gathers slots l, l+32, ... of `buf` (n <= 160): all of its loads are in flight together.
__device__ __forceinline__ u64 poll_min(const u64 *buf, int n, int lane, u64 tag) {
  constexpr int kMaxPer = 5;
  unsigned pending = 0;
  for (int i = 0; i < kMaxPer; ++i) if (lane + 32 * i < n) pending |= 1u << i;
  u64 m = ~0ull;
  while (pending) {
    u64 w0[kMaxPer], w1[kMaxPer];
#pragma unroll
    for (int i = 0; i < kMaxPer; ++i)
      if (pending & (1u << i)) ld_relaxed_v2(buf + (size_t)kSlotStride * (lane + 32 * i), w0[i], w1[i]);
#pragma unroll
    for (int i = 0; i < kMaxPer; ++i)
      if ((pending & (1u << i)) && w1[i] == tag) { pending &= ~(1u << i); m = w0[i] < m ? w0[i] : m; }
  }
  for (int o = 16; o; o >>= 1) { const u64 x = __shfl_xor_sync(0xffffffffu, m, o); m = x < m ? x : m; }
  return m;
}

// ---- l2: flat all-gather through global memory.  PUSH: private row per reader, 32 B slot stride.
template <bool PUSH>
__global__ void __launch_bounds__(32, 1) k_l2(u64 *exch, int S, int rounds, u64 *out) {
  const int lane = threadIdx.x, r = blockIdx.x;
  u64 val = (u64)r + 1;
  for (int g = 0; g < rounds; ++g) {
    const u64 tag = (u64)g + 1;
    u64 m;
    if (PUSH) {
      u64 *buf = exch + (size_t)(g & 1) * S * S * 4;
      for (int d = lane; d < S; d += 32) st_relaxed_v2(buf + ((size_t)d * S + r) * 4, val, tag);
      // own row: S slots of 32 B
      unsigned pending = 0;
      for (int i = 0; i < 5; ++i) if (lane + 32 * i < S) pending |= 1u << i;
      m = ~0ull;
      const u64 *row = buf + (size_t)r * S * 4;
      while (pending) {
        u64 w0[5], w1[5];
#pragma unroll
        for (int i = 0; i < 5; ++i) if (pending & (1u << i)) ld_relaxed_v2(row + (size_t)4 * (lane + 32 * i), w0[i], w1[i]);
#pragma unroll
        for (int i = 0; i < 5; ++i)
          if ((pending & (1u << i)) && w1[i] == tag) { pending &= ~(1u << i); m = w0[i] < m ? w0[i] : m; }
      }
      for (int o = 16; o; o >>= 1) { const u64 x = __shfl_xor_sync(0xffffffffu, m, o); m = x < m ? x : m; }
    } else {
      u64 *buf = exch + (size_t)(g & 1) * S * kSlotStride;
      if (lane == 0) st_relaxed_v2(buf + (size_t)kSlotStride * r, val, tag);
      m = poll_min(buf, S, lane, tag);
    }
    val = m + (u64)r + 1;                      // next round's post depends on this round's result
  }
  if (lane == 0) out[r] = val;
}


// ---- l2near: every poster writes its word to K copies of its slot, kCopyStride bytes apart (so that
// the copies are homed on different L2 partitions / dies with high probability); every CTA first
// measures which copy of each slot it reads fastest and then polls only that one.
constexpr int kCopies = 4;
constexpr size_t kCopyStrideWords = ((size_t)8 << 20) / 8 + 1056;   // 8 MiB + 8448 B, in u64 words
__global__ void __launch_bounds__(32, 1) k_l2near(u64 *exch, int S, int rounds, u64 *out, int calibrate) {
  const int lane = threadIdx.x, r = blockIdx.x;
  // calibration: latency of each copy of the slots this lane polls (min of 8 dependent reads)
  int pick[5] = {0, 0, 0, 0, 0};
  if (calibrate) {
    for (int i = 0; i < 5; ++i) {
      const int s = lane + 32 * i;
      if (s >= S) continue;
      long long best = 1ll << 60;
      for (int c = 0; c < kCopies; ++c) {
        const u64 *p = exch + (size_t)c * kCopyStrideWords + (size_t)kSlotStride * s;
        long long tmin = 1ll << 60;
        for (int rep = 0; rep < 8; ++rep) {
          u64 w0, w1;
          const long long t0 = clock64();
          ld_relaxed_v2(p, w0, w1);
          const long long t1 = clock64() + (long long)(w0 & 0);   // (depends on the load)
          if (t1 - t0 < tmin) tmin = t1 - t0;
        }
        if (tmin < best) { best = tmin; pick[i] = c; }
      }
    }
  }
  __syncwarp();
  u64 val = (u64)r + 1;
  for (int g = 0; g < rounds; ++g) {
    const u64 tag = (u64)g + 1;
    const size_t boff = (size_t)(g & 1) * 256 * kSlotStride;
    if (lane < kCopies)
      st_relaxed_v2(exch + (size_t)lane * kCopyStrideWords + boff + (size_t)kSlotStride * r, val, tag);
    unsigned pending = 0;
    for (int i = 0; i < 5; ++i) if (lane + 32 * i < S) pending |= 1u << i;
    u64 m = ~0ull;
    while (pending) {
      u64 w0[5], w1[5];
#pragma unroll
      for (int i = 0; i < 5; ++i)
        if (pending & (1u << i))
          ld_relaxed_v2(exch + (size_t)pick[i] * kCopyStrideWords + boff + (size_t)kSlotStride * (lane + 32 * i), w0[i], w1[i]);
#pragma unroll
      for (int i = 0; i < 5; ++i)
        if ((pending & (1u << i)) && w1[i] == tag) { pending &= ~(1u << i); m = w0[i] < m ? w0[i] : m; }
    }
    for (int o = 16; o; o >>= 1) { const u64 x = __shfl_xor_sync(0xffffffffu, m, o); m = x < m ? x : m; }
    val = m + (u64)r + 1;
  }
  if (lane == 0) out[r] = val;
}


// ---- l2die: the CTAs are split into two groups by SM id (< 74 or not: the two dies, if SM ids are
// laid out that way) and each group all-gathers on its own slots: does locality lower the floor?
// GROUPING 0: by SM id half; 1: by SM id parity (a control: same group sizes, no locality).
template <int GROUPING>
__global__ void __launch_bounds__(32, 1) k_l2die(u64 *exch, unsigned *counters, int rounds, u64 *out) {
  const int lane = threadIdx.x;
  unsigned smid;
  asm volatile("mov.u32 %0, %%smid;" : "=r"(smid));
  const int grp = GROUPING == 0 ? (smid >= 74u ? 1 : 0) : (int)(smid & 1u);
  __shared__ int s_rank, s_size;
  if (lane == 0) s_rank = (int)atomicAdd(&counters[grp], 1u);
  __syncwarp();
  cooperative_groups::this_grid().sync();
  if (lane == 0) s_size = (int)counters[grp];
  __syncwarp();
  const int r = s_rank, S = s_size;
  u64 *base = exch + (size_t)grp * 2 * 256 * kSlotStride;
  u64 val = (u64)blockIdx.x + 1;
  for (int g = 0; g < rounds; ++g) {
    const u64 tag = (u64)g + 1;
    u64 *buf = base + (size_t)(g & 1) * 256 * kSlotStride;
    if (lane == 0) st_relaxed_v2(buf + (size_t)kSlotStride * r, val, tag);
    const u64 m = poll_min(buf, S, lane, tag);
    val = m + (u64)blockIdx.x + 1;
  }
  if (lane == 0) out[blockIdx.x] = val + (u64)S;
}

// ---- MODE 0 dsmem, 1 hybrid (all poll), 2 hyblead (leaders poll, DSMEM broadcast), 3 hybpush
template <int MODE>
__global__ void __launch_bounds__(32, 1) k_cluster(u64 *exch, int C, int n_clusters, int rounds, u64 *out) {
  extern __shared__ __align__(16) unsigned char dyn[];   // (sized like the product's state, unused)
  __shared__ __align__(16) u64 slots[2][16][2];
  __shared__ __align__(16) u64 result[2][2];
  __shared__ __align__(8) u64 bars[2], bars2[2];
  const int lane = threadIdx.x;
  const uint32_t cr = cluster_rank();
  const int cl = blockIdx.x / C;
  const int n_ctas = C * n_clusters;
  if (lane == 0) {
    mbar_init(smem_addr(&bars[0]), 1); mbar_init(smem_addr(&bars[1]), 1);
    mbar_init(smem_addr(&bars2[0]), 1); mbar_init(smem_addr(&bars2[1]), 1);
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
  }
  cluster_sync_all();
  u64 val = (u64)blockIdx.x + 1;
  for (int g = 0; g < rounds; ++g) {
    const int par = g & 1;
    const uint32_t ph = (uint32_t)((g >> 1) & 1);
    const uint32_t bar = smem_addr(&bars[par]);
    if (lane == 0) mbar_expect_tx(bar, 16u * (uint32_t)C);
    if (lane < C)
      st_async_v2(mapa(smem_addr(&slots[par][cr][0]), (uint32_t)lane), val, (u64)g, mapa(bar, (uint32_t)lane));
    while (!mbar_try_wait(bar, ph)) {}
    u64 m = (lane < C) ? slots[par][lane][0] : ~0ull;
    for (int o = 16; o; o >>= 1) { const u64 x = __shfl_xor_sync(0xffffffffu, m, o); m = x < m ? x : m; }
    const u64 tag = (u64)g + 1;
    if (MODE == 1) {
      u64 *buf = exch + (size_t)par * n_clusters * kSlotStride;
      if (cr == 0 && lane == 0) st_relaxed_v2(buf + (size_t)kSlotStride * cl, m, tag);
      m = poll_min(buf, n_clusters, lane, tag);
    } else if (MODE == 2) {
      const uint32_t bar2 = smem_addr(&bars2[par]);
      if (lane == 0) mbar_expect_tx(bar2, 16u);
      if (cr == 0) {
        u64 *buf = exch + (size_t)par * n_clusters * kSlotStride;
        if (lane == 0) st_relaxed_v2(buf + (size_t)kSlotStride * cl, m, tag);
        m = poll_min(buf, n_clusters, lane, tag);
        if (lane < C) st_async_v2(mapa(smem_addr(&result[par][0]), (uint32_t)lane), m, tag, mapa(bar2, (uint32_t)lane));
      }
      while (!mbar_try_wait(bar2, ph)) {}
      m = result[par][0];
    } else if (MODE == 3) {
      u64 *buf = exch + (size_t)par * n_ctas * n_clusters * 4;
      if (cr == 0)
        for (int d = lane; d < n_ctas; d += 32) st_relaxed_v2(buf + ((size_t)d * n_clusters + cl) * 4, m, tag);
      const u64 *row = buf + (size_t)blockIdx.x * n_clusters * 4;
      unsigned pending = 0;
      for (int i = 0; i < 3; ++i) if (lane + 32 * i < n_clusters) pending |= 1u << i;
      m = ~0ull;
      while (pending) {
        u64 w0[3], w1[3];
#pragma unroll
        for (int i = 0; i < 3; ++i) if (pending & (1u << i)) ld_relaxed_v2(row + (size_t)4 * (lane + 32 * i), w0[i], w1[i]);
#pragma unroll
        for (int i = 0; i < 3; ++i)
          if ((pending & (1u << i)) && w1[i] == tag) { pending &= ~(1u << i); m = w0[i] < m ? w0[i] : m; }
      }
      for (int o = 16; o; o >>= 1) { const u64 x = __shfl_xor_sync(0xffffffffu, m, o); m = x < m ? x : m; }
    }
    val = m + (u64)blockIdx.x + 1;
  }
  if (lane == 0) out[blockIdx.x] = val;
  cluster_sync_all();                          // no CTA exits while a peer may still write to it
}

static float time_launch(cudaLaunchConfig_t &cfg, const void *fn, void **args) {
  cudaEvent_t e0, e1;
  CK(cudaEventCreate(&e0)); CK(cudaEventCreate(&e1));
  CK(cudaLaunchKernelExC(&cfg, fn, args));     // warm-up
  CK(cudaDeviceSynchronize());
  CK(cudaEventRecord(e0));
  CK(cudaLaunchKernelExC(&cfg, fn, args));
  CK(cudaEventRecord(e1));
  CK(cudaDeviceSynchronize());
  float ms; CK(cudaEventElapsedTime(&ms, e0, e1));
  return ms;
}

template <int MODE>
static void run_cluster_mode(const char *name, int C, int ncl, size_t dyn, u64 *exch, size_t exch_bytes, u64 *out, int rounds) {
  const void *fn = (const void *)k_cluster<MODE>;
  CK(cudaFuncSetAttribute(fn, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)dyn));
  CK(cudaFuncSetAttribute(fn, cudaFuncAttributeNonPortableClusterSizeAllowed, 1));
  cudaLaunchConfig_t cfg = {};
  cfg.blockDim = dim3(32); cfg.dynamicSmemBytes = dyn; cfg.gridDim = dim3(C * ncl);
  cudaLaunchAttribute at[2];
  at[0].id = cudaLaunchAttributeClusterDimension;
  at[0].val.clusterDim.x = C; at[0].val.clusterDim.y = 1; at[0].val.clusterDim.z = 1;
  at[1].id = cudaLaunchAttributeCooperative; at[1].val.cooperative = 1;
  cfg.attrs = at; cfg.numAttrs = MODE == 0 ? 1 : 2;   // clusters that spin on one another: cooperative
  void *args[] = {&exch, &C, &ncl, &rounds, &out};
  float best = 1e30f;
  for (int rep = 0; rep < 3; ++rep) {
    CK(cudaMemset(exch, 0, exch_bytes));
    cudaEvent_t e0, e1;
    CK(cudaEventCreate(&e0)); CK(cudaEventCreate(&e1));
    CK(cudaEventRecord(e0));
    cudaError_t le = cudaLaunchKernelExC(&cfg, fn, args);
    if (le != cudaSuccess) { printf("%s,%d,%d,%d,launch refused (%s)\n", name, C * ncl, C, ncl, cudaGetErrorString(le)); cudaGetLastError(); return; }
    CK(cudaEventRecord(e1));
    CK(cudaDeviceSynchronize());
    float ms; CK(cudaEventElapsedTime(&ms, e0, e1));
    if (rep > 0 && ms < best) best = ms;
  }
  printf("%s,%d,%d,%d,%.3f\n", name, C * ncl, C, ncl, best * 1e3 / rounds);
}

int main() {
  int rounds = 20000;
  u64 *exch, *out;
  const size_t exch_bytes = (size_t)kCopies * kCopyStrideWords * 8 + ((size_t)1 << 20);   // (covers every variant)
  CK(cudaMalloc(&exch, exch_bytes));
  CK(cudaMalloc(&out, 256 * 8));
  const size_t dyn = 200 * 1024;               // like the product: one CTA per SM

  printf("mode,ctas,cluster,n_clusters,us_per_round\n");
  for (int push = 0; push < 2; ++push)
    for (int S : {1, 2, 4, 8, 16, 37, 74, 96, 128, 148}) {
      cudaLaunchConfig_t cfg = {};
      const void *fn = push ? (const void *)k_l2<true> : (const void *)k_l2<false>;
      CK(cudaFuncSetAttribute(fn, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)dyn));
      cfg.gridDim = dim3(S); cfg.blockDim = dim3(32); cfg.dynamicSmemBytes = dyn;   // one CTA per SM
      cudaLaunchAttribute at[1];
      at[0].id = cudaLaunchAttributeCooperative; at[0].val.cooperative = 1;
      cfg.attrs = at; cfg.numAttrs = 1;
      void *args[] = {&exch, &S, &rounds, &out};
      float best = 1e30f;
      for (int rep = 0; rep < 3; ++rep) {
        CK(cudaMemset(exch, 0, exch_bytes));
        const float ms = time_launch(cfg, push ? (const void *)k_l2<true> : (const void *)k_l2<false>, args);
        if (ms < best) best = ms;
      }
      printf("%s,%d,1,%d,%.3f\n", push ? "l2push" : "l2", S, S, best * 1e3 / rounds);
    }
  for (int cal = 0; cal < 2; ++cal)
    for (int S : {16, 37, 74, 148}) {
      cudaLaunchConfig_t cfg = {};
      cfg.gridDim = dim3(S); cfg.blockDim = dim3(32); cfg.dynamicSmemBytes = 0;
      cudaLaunchAttribute at[1];
      at[0].id = cudaLaunchAttributeCooperative; at[0].val.cooperative = 1;
      cfg.attrs = at; cfg.numAttrs = 1;
      void *args[] = {&exch, &S, &rounds, &out, &cal};
      float best = 1e30f;
      for (int rep = 0; rep < 3; ++rep) {
        CK(cudaMemset(exch, 0, exch_bytes));
        const float ms = time_launch(cfg, (const void *)k_l2near, args);
        if (ms < best) best = ms;
      }
      printf("%s,%d,1,%d,%.3f\n", cal ? "l2near" : "l2copies", S, S, best * 1e3 / rounds);
    }
  for (int grouping = 0; grouping < 2; ++grouping) {
    unsigned *counters;
    CK(cudaMalloc(&counters, 8));
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = dim3(148); cfg.blockDim = dim3(32); cfg.dynamicSmemBytes = 0;
    cudaLaunchAttribute at[1];
    at[0].id = cudaLaunchAttributeCooperative; at[0].val.cooperative = 1;
    cfg.attrs = at; cfg.numAttrs = 1;
    void *args[] = {&exch, &counters, &rounds, &out};
    float best = 1e30f;
    for (int rep = 0; rep < 3; ++rep) {
      CK(cudaMemset(exch, 0, exch_bytes));
      CK(cudaMemset(counters, 0, 8));
      cudaEvent_t e0, e1;
      CK(cudaEventCreate(&e0)); CK(cudaEventCreate(&e1));
      CK(cudaEventRecord(e0));
      CK(cudaLaunchKernelExC(&cfg, grouping ? (const void *)k_l2die<1> : (const void *)k_l2die<0>, args));
      CK(cudaEventRecord(e1));
      CK(cudaDeviceSynchronize());
      float ms; CK(cudaEventElapsedTime(&ms, e0, e1));
      if (ms < best) best = ms;
    }
    printf("%s,148,1,2,%.3f\n", grouping ? "l2parity" : "l2die", best * 1e3 / rounds);
  }
  for (int C : {2, 4, 6, 8, 16}) {
    cudaLaunchConfig_t cfg = {};
    cfg.blockDim = dim3(32); cfg.dynamicSmemBytes = dyn;
    cudaLaunchAttribute at[1];
    at[0].id = cudaLaunchAttributeClusterDimension;
    at[0].val.clusterDim.x = C; at[0].val.clusterDim.y = 1; at[0].val.clusterDim.z = 1;
    cfg.attrs = at; cfg.numAttrs = 1;
    cfg.gridDim = dim3(C);
    CK(cudaFuncSetAttribute(k_cluster<0>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)dyn));
    CK(cudaFuncSetAttribute(k_cluster<0>, cudaFuncAttributeNonPortableClusterSizeAllowed, 1));
    int max_clusters = 0;
    cudaError_t e = cudaOccupancyMaxActiveClusters(&max_clusters, (const void *)k_cluster<0>, &cfg);
    if (e != cudaSuccess) { printf("dsmem,%d,%d,0,unsupported (%s)\n", C, C, cudaGetErrorString(e)); cudaGetLastError(); continue; }
    printf("# cluster size %d with %zu KB dynamic shared memory: %d clusters co-resident\n", C, dyn / 1024, max_clusters);
    if (max_clusters < 1) continue;
    run_cluster_mode<0>("dsmem", C, 1, dyn, exch, exch_bytes, out, rounds);
    run_cluster_mode<0>("dsmem", C, max_clusters, dyn, exch, exch_bytes, out, rounds);
    run_cluster_mode<1>("hybrid", C, max_clusters, dyn, exch, exch_bytes, out, rounds);
    run_cluster_mode<2>("hyblead", C, max_clusters, dyn, exch, exch_bytes, out, rounds);
    run_cluster_mode<3>("hybpush", C, max_clusters, dyn, exch, exch_bytes, out, rounds);
  }
  return 0;
}
