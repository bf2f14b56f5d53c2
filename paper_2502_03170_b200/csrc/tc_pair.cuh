// CTA-pair (cta_group::2) versions of the two tcgen05 stages for the 3xFP16 path.  Two CTAs on the SMs of one TPC form a
// cluster and execute each UMMA together: M = 256 rows (128 per CTA), N = 256 columns of which each CTA stages one half
// (128 rows of the B operand).  Per CTA this halves the B-operand bytes per flop: the L2 -> SM ingress and the
// shared-memory read bandwidth stop being the limit they are for single-CTA 128 x 256 tiles with hi + lo operands
// (DESIGN.md §5).  Only the leader CTA (cluster rank 0) issues tcgen05.mma; both CTAs load / generate operands, both
// drain their own 128 TMEM lanes.
//
//   k1_pair (stage 1):  D[mx, (half, slot, ql)] = X_g[mx, qx] * Q[(half, slot, ql), qx]^T      M = 256 mx, N = 256
//       A = cos / sin table rows of the CTA's own 128 mx, by TMA;
//       B = pupil field: CTA `half` generates slots (4 chains of the x-parity group) x 32 q_y = 128 rows straight into its
//           swizzled shared memory (each pupil element is generated once per pair); the base pupil of a stage arrives by
//           one bulk copy into a shared-memory ring, the defocus phasors of a tile live in registers;
//       epilogue: one thread per mx row holds 64 consecutive q_y of a chain -> scale, fp16 hi / lo, 16-byte stores into a
//           swizzled staging tile, TMA store into T^T[chain][mx][qy].
//   k2_pair (stage 2):  D[my, (slot, mx)] = Y_a[my, qy] * T^T[(slot, mx), qy]^T                 M = 256 my, N = 4 x 64
//       both operands by TMA (each CTA: its own 128 my rows of the table, 2 of the 4 chains of T^T);
//       epilogue as k2_tc (mirror butterfly, |E|^2, running sums over the components) with a coalesced final store
//       through a padded shared-memory tile.
#pragma once
#include <cuda.h>
#include <cuda_fp16.h>

#include "pupil_gen.cuh"
#include "tc_common.cuh"

namespace psf {
namespace pair {

using namespace tc;

// ---- cluster / pair primitives ---------------------------------------------------------------------------------------
__device__ __forceinline__ uint32_t cluster_ctarank() {
  uint32_t r;
  asm volatile("mov.u32 %0, %%cluster_ctarank;" : "=r"(r));
  return r;
}
__device__ __forceinline__ void cluster_sync_all() {
  asm volatile("barrier.cluster.arrive.release.aligned;" ::: "memory");
  asm volatile("barrier.cluster.wait.acquire.aligned;" ::: "memory");
}
// shared::cluster address of `saddr` (a shared::cta address of this CTA) in CTA `rank` of the cluster
__device__ __forceinline__ uint32_t mapa(uint32_t saddr, uint32_t rank) {
  uint32_t r;
  asm volatile("mapa.shared::cluster.u32 %0, %1, %2;" : "=r"(r) : "r"(saddr), "r"(rank));
  return r;
}
// default semantics (release at CTA scope): a cluster-scope release compiles to MEMBAR.ALL.GPU + ERRBAR, microseconds per
// arrive, and is not needed: accumulator hand-backs carry no memory data (TMEM reads completed by tcgen05.wait::ld +
// tcgen05.fence), and the stage-1 operand rows are fenced for the async proxy inside their own CTA before the signal.
__device__ __forceinline__ void mbar_arrive_cluster(uint32_t cluster_addr) {
  asm volatile("mbarrier.arrive.shared::cluster.b64 _, [%0];" ::"r"(cluster_addr) : "memory");
}
// cluster-scope release: every write this thread has observed (its own and, cumulatively, those it acquired) is performed
// with respect to the whole cluster before the arrive becomes visible (SASS: MEMBAR.ALL.GPU + ERRBAR ahead of the arrive)
__device__ __forceinline__ void mbar_arrive_cluster_release(uint32_t cluster_addr) {
  asm volatile("mbarrier.arrive.release.cluster.shared::cluster.b64 _, [%0];" ::"r"(cluster_addr) : "memory");
}
__device__ __forceinline__ void mbar_wait_acquire_cluster(uint64_t *bar, uint32_t parity) {
  uint32_t ok;
  do {
    asm volatile(
        "{\n\t.reg .pred p;\n\tmbarrier.try_wait.parity.acquire.cluster.shared::cta.b64 p, [%1], %2;\n\tselp.u32 %0, 1, 0, p;\n\t}"
        : "=r"(ok)
        : "r"(smem_u32(bar)), "r"(parity)
        : "memory");
  } while (!ok);
}
template <int N> __device__ __forceinline__ void setmaxnreg_inc() { asm volatile("setmaxnreg.inc.sync.aligned.u32 %0;" ::"n"(N)); }
template <int N> __device__ __forceinline__ void setmaxnreg_dec() { asm volatile("setmaxnreg.dec.sync.aligned.u32 %0;" ::"n"(N)); }
// (waits use the plain mbar_wait: an .acquire.cluster try_wait adds an L1 invalidate, CCTL.IVALL, to every successful wait)
// TMA loads whose completion bytes are credited to an mbarrier of the pair's leader CTA (`bar_cluster` = mapa(bar, 0))
__device__ __forceinline__ void tma2_load_2d(uint32_t smem_dst, const void *tmap, uint32_t bar_cluster, int x, int y) {
  asm volatile(
      "cp.async.bulk.tensor.2d.cta_group::2.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1, {%3, %4}], [%2];"
      ::"r"(smem_dst), "l"((uint64_t)tmap), "r"(bar_cluster), "r"(x), "r"(y)
      : "memory");
}
__device__ __forceinline__ void tma2_load_3d(uint32_t smem_dst, const void *tmap, uint32_t bar_cluster, int x, int y, int z) {
  asm volatile(
      "cp.async.bulk.tensor.3d.cta_group::2.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1, {%3, %4, %5}], [%2];"
      ::"r"(smem_dst), "l"((uint64_t)tmap), "r"(bar_cluster), "r"(x), "r"(y), "r"(z)
      : "memory");
}
// TMA store shared -> global (bulk async-group completion)
__device__ __forceinline__ void tma_store_3d(const void *tmap, uint32_t smem_src, int x, int y, int z) {
  asm volatile("cp.async.bulk.tensor.3d.global.shared::cta.bulk_group [%0, {%2, %3, %4}], [%1];"
               ::"l"((uint64_t)tmap), "r"(smem_src), "r"(x), "r"(y), "r"(z)
               : "memory");
}
__device__ __forceinline__ void bulk_commit() { asm volatile("cp.async.bulk.commit_group;" ::: "memory"); }
template <int N>
__device__ __forceinline__ void bulk_wait_read() { asm volatile("cp.async.bulk.wait_group.read %0;" ::"n"(N) : "memory"); }
__device__ __forceinline__ void bulk_wait_all() { asm volatile("cp.async.bulk.wait_group 0;" ::: "memory"); }

__device__ __forceinline__ void tmem_alloc2(uint32_t *slot, uint32_t cols) {
  asm volatile("tcgen05.alloc.cta_group::2.sync.aligned.shared::cta.b32 [%0], %1;" ::"r"(smem_u32(slot)), "r"(cols) : "memory");
  asm volatile("tcgen05.relinquish_alloc_permit.cta_group::2.sync.aligned;" ::: "memory");
}
__device__ __forceinline__ void tmem_dealloc2(uint32_t base, uint32_t cols) {
  asm volatile("tcgen05.dealloc.cta_group::2.sync.aligned.b32 %0, %1;" ::"r"(base), "r"(cols) : "memory");
}
__device__ __forceinline__ void umma2_f16(uint32_t d_tmem, uint64_t a_desc, uint64_t b_desc, uint32_t idesc, uint32_t accumulate) {
  asm volatile(
      "{\n\t.reg .pred p;\n\tsetp.ne.b32 p, %4, 0;\n\t"
      "tcgen05.mma.cta_group::2.kind::f16 [%0], %1, %2, %3, p;\n\t}"
      ::"r"(d_tmem), "l"(a_desc), "l"(b_desc), "r"(idesc), "r"(accumulate)
      : "memory");
}
// arrive on the barrier at the same shared-memory offset in both CTAs once the pair's previously issued UMMAs are done
__device__ __forceinline__ void umma2_commit(uint64_t *bar, uint16_t cta_mask = 3) {
  asm volatile("tcgen05.commit.cta_group::2.mbarrier::arrive::one.shared::cluster.multicast::cluster.b64 [%0], %1;"
               ::"r"(smem_u32(bar)), "h"(cta_mask)
               : "memory");
}
__device__ __forceinline__ void named_bar_sync(int id, int nthreads) {
  asm volatile("bar.sync %0, %1;" ::"r"(id), "r"(nthreads) : "memory");
}
__device__ __forceinline__ void st_shared_v4(uint32_t saddr, uint32_t a, uint32_t b, uint32_t c, uint32_t d) {
  asm volatile("st.shared.v4.b32 [%0], {%1, %2, %3, %4};" ::"r"(saddr), "r"(a), "r"(b), "r"(c), "r"(d) : "memory");
}

constexpr int TILE16K = 128 * 128;                       // 128 rows x one 128-byte swizzle row
constexpr int P_STAGE = 4 * TILE16K;                     // A hi, A lo, B-half hi, B-half lo = 64 KB per CTA
constexpr uint32_t P_IDESC = umma_idesc_f16(256, 256);

// one K = 16 step of a stage: D += A_lo B_hi + A_hi B_lo + A_hi B_hi
__device__ __forceinline__ void issue_kstep2(uint32_t sbase, uint32_t d_tmem, int k, bool zero) {
  const uint32_t ah = sbase, al = sbase + TILE16K, bh = sbase + 2 * TILE16K, bl = sbase + 3 * TILE16K;
  const uint32_t o = k * 32;
  umma2_f16(d_tmem, umma_desc_sw128(al + o), umma_desc_sw128(bh + o), P_IDESC, zero ? 0u : 1u);
  umma2_f16(d_tmem, umma_desc_sw128(ah + o), umma_desc_sw128(bl + o), P_IDESC, 1u);
  umma2_f16(d_tmem, umma_desc_sw128(ah + o), umma_desc_sw128(bh + o), P_IDESC, 1u);
}
// one stage = 64 contraction indices = four K = 16 steps
__device__ __forceinline__ void issue_stage_mmas2(uint32_t sbase, uint32_t d_tmem, bool first) {
#pragma unroll
  for (int k = 0; k < 4; ++k) issue_kstep2(sbase, d_tmem, k, first && k == 0);
}

// ---- stage 2 ----------------------------------------------------------------------------------------------------------
struct K2PArgs {
  float *intensity;     // [Z][M][M]
  float2 *field;        // [C][Z][M][M] or nullptr (FIELD kernels only)
  int C, n_pad, m_pad, m, M, z0, zc, Z;
  float weight[5];      // intensity weights times the inverse operand scales squared
  float fscale;         // 1 / (s_X s_T): accumulator -> field
};

// ---- fused launch (k12_fused): both stages in one persistent kernel, stage-2 clusters consuming T^T right behind the stage-1
// clusters that produce it, so that the hand-off scratch is a small ring that stays in L2 instead of a 2.7 GB round trip
// through HBM (config 5).  Global flags carry the dependencies:
//   ready[z C + c]    += 1 by each stage-1 CTA whose TMA stores of (plane z, component c) have completed   (target 2 a1)
//   consumed[z C + c] += 1 by each stage-2 cluster whose TMA loads of (plane z, component c) have landed  (target a2)
// Clusters are scheduled round-robin over tiles, a1 (a2) consecutive stage-1 (stage-2) tiles per plane, n1 = Pg a1 stage-1
// clusters and Pg a2 stage-2 clusters: Pg planes are in flight, plane z belongs to group z % Pg, and the (plane, component)
// units of a group rotate through U ring slots of the scratch.  Everything is resident at once (one cluster per SM pair),
// so the spins cannot deadlock; a spin that runs out sets `abort`, after which nobody waits (the results are then wrong and
// the host reports it, but the launch ends).
struct FuseCtx {
  int *ready, *consumed, *abort;
  int n1, a1, a2, Pg, U;
};
struct FuseUnit { int ring, prev; };     // ring unit of (plane, component); flag index of the unit that used the slot before (-1: none)
__device__ __forceinline__ FuseUnit fuse_unit(const FuseCtx &F, int C, int zl, int c) {
  const int gi = zl % F.Pg, k = zl / F.Pg;
  const int i = k * C + c;
  FuseUnit u;
  u.ring = gi * F.U + i % F.U;
  const int ip = i - F.U;
  u.prev = ip < 0 ? -1 : (gi + (ip / C) * F.Pg) * C + ip % C;
  return u;
}
// (the abort word is in mapped host memory: polled every 4096 spins only)
__device__ __forceinline__ int ld_acquire_gpu(const int *p) {
  int v;
  asm volatile("ld.acquire.gpu.global.s32 %0, [%1];" : "=r"(v) : "l"(p) : "memory");
  return v;
}
__device__ __forceinline__ void red_release_gpu_add(int *p, int v) {
  asm volatile("red.release.gpu.global.add.s32 [%0], %1;" ::"l"(p), "r"(v) : "memory");
}
__device__ __forceinline__ void fence_proxy_async_all() { asm volatile("fence.proxy.async;" ::: "memory"); }
__device__ __forceinline__ void fuse_wait(const FuseCtx &F, const int *flag, int target) {
  unsigned spins = 0;
  while (ld_acquire_gpu(flag) < target) {
    __nanosleep(40);
    if ((++spins & 0xFFFu) == 0) {
      if (*(volatile int *)F.abort) break;
      if (spins > (1u << 24)) { atomicExch_system(F.abort, 1); break; }   // ~1 s: something is wrong; stop waiting everywhere
    }
  }
}
template <int N>
__device__ __forceinline__ void bulk_wait_complete() { asm volatile("cp.async.bulk.wait_group %0;" ::"n"(N) : "memory"); }

constexpr int K2P_NST = 3;
constexpr int K2P_EPI_WARPS = 16;
constexpr int K2P_THREADS = 32 * (4 + K2P_EPI_WARPS);
constexpr int K2P_PITCH = 65;                                    // staging row pitch in floats (conflict-free column writes)
constexpr int K2P_STAGING = 128 * K2P_PITCH * 4;
constexpr int K2P_SMEM = 1024 + K2P_NST * P_STAGE + K2P_STAGING;

struct K2PShared {
  uint64_t full[K2P_NST], empty[K2P_NST], acc_full, acc_empty;
  uint32_t tmem_slot;
};

// TMA warp (both CTAs) and MMA warp (leader CTA)
template <bool FUSED>
__device__ __forceinline__ void k2p_feed(uint8_t *smem, K2PShared &S, uint32_t tmem, const CUtensorMap &map_xhi, const CUtensorMap &map_xlo,
                                         const CUtensorMap &map_thi, const CUtensorMap &map_tlo, const K2PArgs &P, int warp, uint32_t rank,
                                         int nk, int tiles_yp, int tiles_x, int ntiles, int ncl, int cid, const FuseCtx &F) {
  const bool leader = rank == 0;
  uint64_t *full = S.full, *empty = S.empty;
  uint64_t &acc_full = S.acc_full, &acc_empty = S.acc_empty;
  if (warp == 0) {
    // ---------------- TMA: own 128 table rows (A) and 2 of the 4 chains of T^T (B half) ----------------
    if (elect_one()) {
      int st = 0, ph = 0;
      uint32_t full_leader[K2P_NST];
      for (int i = 0; i < K2P_NST; ++i) full_leader[i] = mapa(smem_u32(&full[i]), 0);
      if (!FUSED) tc::pdl_wait();                          // two-kernel path: T^T is the stage-1 grid's output
      for (int t = cid; t < ntiles; t += ncl) {
        const int typ = t % tiles_yp;
        int r = t / tiles_yp;
        const int tx = r % tiles_x;
        const int zl = r / tiles_x;
        const int ty = typ * 2 + (int)rank;
        for (int c = 0; c < P.C; ++c) {
          int unit = zl * P.C + c;
          if (FUSED) {                                     // T^T of (plane, component) is complete in the ring scratch
            unit = fuse_unit(F, P.C, zl, c).ring;
            fuse_wait(F, F.ready + zl * P.C + c, 2 * F.a1);
            fence_proxy_async_all();                       // the TMA reads below are ordered behind the acquire
          }
          for (int a = 0; a < 2; ++a) {
            const int arow = a * P.m_pad + ty * 128;
            const int chain0 = unit * 8 + 4 * a + 2 * (int)rank;
            for (int kc = 0; kc < nk; ++kc) {
              mbar_wait(&empty[st], ph ^ 1);
              const uint32_t s = smem_u32(smem + st * P_STAGE);
              if (leader) mbar_arrive_expect_tx(&full[st], 2 * P_STAGE);
              tma2_load_2d(s, &map_xhi, full_leader[st], kc * 64, arow);
              tma2_load_2d(s + TILE16K, &map_xlo, full_leader[st], kc * 64, arow);
              tma2_load_3d(s + 2 * TILE16K, &map_thi, full_leader[st], kc * 64, tx * 64, chain0);
              tma2_load_3d(s + 3 * TILE16K, &map_tlo, full_leader[st], kc * 64, tx * 64, chain0);
              if (++st == K2P_NST) { st = 0; ph ^= 1; }
            }
          }
        }
      }
    }
  } else if (warp == 1) {
    // ---------------- MMA issuer (leader CTA only) ----------------
    if (leader && elect_one()) {
      int st = 0, ph = 0, item = 0;
      for (int t = cid; t < ntiles; t += ncl) {
        for (int c = 0; c < P.C; ++c, ++item) {
          mbar_wait(&acc_empty, (item & 1) ^ 1);
          tcgen05_fence_after();
          for (int a = 0; a < 2; ++a) {
            const uint32_t d = tmem + a * 256;
            for (int kc = 0; kc < nk; ++kc) {
              mbar_wait(&full[st], ph);
              tcgen05_fence_after();
              issue_stage_mmas2(smem_u32(smem + st * P_STAGE), d, kc == 0);
              umma2_commit(&empty[st]);
              if (++st == K2P_NST) { st = 0; ph ^= 1; }
            }
          }
          if (FUSED) {                                     // every T^T tile of (plane, component) has landed in the pair's shared memory
            const int zl = (t / tiles_yp) / tiles_x;
            red_release_gpu_add(F.consumed + zl * P.C + c, 1);
          }
          umma2_commit(&acc_full);
        }
      }
    }
  }
}

// Field store of one group of four consecutive m_x of every row of a warp (warp-collective).  v[quadrant][u] = E at the four
// mirror images of pixel (row, mxg + u).  vec (M a multiple of 8): two lanes share a row so that one STG.128 of the warp
// writes full 32-byte sectors (16 rows x 32 contiguous bytes) - the halves travel by shuffle; else 8-byte stores per pixel.
__device__ __forceinline__ void store_field_group(float2 *f, int M, int m, int row0, int lane, int mxg, const float2 (&v)[4][4], float fs, bool vec) {
  if (!vec) {
    const int my = row0 + lane;
    if (my < m) {
#pragma unroll
      for (int u = 0; u < 4; ++u) {
        const int mx = mxg + u;
        if (mx < m) {
          const int myr = M - 1 - my, mxr = M - 1 - mx;
          f[(size_t)my * M + mx] = make_float2(fs * v[0][u].x, fs * v[0][u].y);
          f[(size_t)my * M + mxr] = make_float2(fs * v[1][u].x, fs * v[1][u].y);
          f[(size_t)myr * M + mx] = make_float2(fs * v[2][u].x, fs * v[2][u].y);
          f[(size_t)myr * M + mxr] = make_float2(fs * v[3][u].x, fs * v[3][u].y);
        }
      }
    }
    return;
  }
  const int odd = lane & 1;
#pragma unroll
  for (int qd = 0; qd < 4; ++qd) {
    const bool mirx = qd & 1;
    // the 32-byte block of the group in ascending address order: low half, high half
    const float4 low = mirx ? make_float4(v[qd][3].x, v[qd][3].y, v[qd][2].x, v[qd][2].y) : make_float4(v[qd][0].x, v[qd][0].y, v[qd][1].x, v[qd][1].y);
    const float4 high = mirx ? make_float4(v[qd][1].x, v[qd][1].y, v[qd][0].x, v[qd][0].y) : make_float4(v[qd][2].x, v[qd][2].y, v[qd][3].x, v[qd][3].y);
    const float4 send = odd ? low : high;
    float4 recv;
    recv.x = __shfl_xor_sync(0xffffffffu, send.x, 1); recv.y = __shfl_xor_sync(0xffffffffu, send.y, 1);
    recv.z = __shfl_xor_sync(0xffffffffu, send.z, 1); recv.w = __shfl_xor_sync(0xffffffffu, send.w, 1);
    const int col = (mirx ? M - 4 - mxg : mxg) + 2 * odd;
    if (mxg < m) {
#pragma unroll
      for (int k = 0; k < 2; ++k) {                   // k = 0: the even row of the lane pair, k = 1: the odd row
        const int my = row0 + (lane & ~1) + k;
        if (my < m) {
          const float4 val = k == 0 ? (odd ? recv : low) : (odd ? high : recv);
          const int y = (qd & 2) ? M - 1 - my : my;
          *reinterpret_cast<float4 *>(f + (size_t)y * M + col) = make_float4(fs * val.x, fs * val.y, fs * val.z, fs * val.w);
        }
      }
    }
  }
}

// sixteen epilogue warps: butterfly + |E|^2, running sums over the components, coalesced quadrant stores
// (FIELD: the four mirror values of E_c are also stored, 32 bytes per thread and store, straight from the registers)
template <bool FIELD>
__device__ __forceinline__ void k2p_epilogue(float *staging, K2PShared &S, uint32_t tmem, const K2PArgs &P, int warp, int lane, uint32_t rank,
                                             int tiles_yp, int tiles_x, int ntiles, int ncl, int cid) {
  uint64_t &acc_full = S.acc_full, &acc_empty = S.acc_empty;
  {
    const int q = warp & 3;                 // TMEM lane quarter
    const int e = (warp - 4) >> 2;          // 16-column slice of the 64 mx of the tile
    const int wi = warp - 4;
    const uint32_t acc_empty_leader = mapa(smem_u32(&acc_empty), 0);
    int item = 0;
    for (int t = cid; t < ntiles; t += ncl) {
      const int typ = t % tiles_yp;
      int r = t / tiles_yp;
      const int tx = r % tiles_x;
      const int zl = r / tiles_x;
      const int ty = typ * 2 + (int)rank;
      float sum[4][16];
#pragma unroll
      for (int qd = 0; qd < 4; ++qd)
#pragma unroll
        for (int i = 0; i < 16; ++i) sum[qd][i] = 0.f;
      for (int c = 0; c < P.C; ++c, ++item) {
        const float w = P.weight[c];
        mbar_wait(&acc_full, item & 1);
        tcgen05_fence_after();
#pragma unroll
        for (int i4 = 0; i4 < 4; ++i4) {
          uint32_t v[8][4];
#pragma unroll
          for (int ch = 0; ch < 8; ++ch)
            tmem_ld_32x32b_x4(tmem + ((uint32_t)(q * 32) << 16) + (ch >> 2) * 256 + (ch & 3) * 64 + e * 16 + i4 * 4, v[ch]);
          tmem_ld_wait();
          if (i4 == 3) {                      // every TMEM read of this item is done: the MMAs of the next one may start
            tcgen05_fence_before();
            __syncwarp();
            if (lane == 0) mbar_arrive_cluster(acc_empty_leader);
          }
          float2 fe[FIELD ? 4 : 1][FIELD ? 4 : 1];
#pragma unroll
          for (int u = 0; u < 4; ++u) {
            const float a0 = __uint_as_float(v[0][u]), a1 = __uint_as_float(v[1][u]), a2 = __uint_as_float(v[2][u]),
                        a3 = __uint_as_float(v[3][u]), a4 = __uint_as_float(v[4][u]), a5 = __uint_as_float(v[5][u]),
                        a6 = __uint_as_float(v[6][u]), a7 = __uint_as_float(v[7][u]);
            const float pr = a0 - a5, qr = a0 + a5, rr = a3 + a6, sr = a3 - a6;
            const float pi = a1 + a4, qi = a1 - a4, ri = a2 - a7, si = a2 + a7;
            const float re0 = pr - rr, im0 = pi + ri;   // (my, mx)
            const float re1 = pr + rr, im1 = pi - ri;   // (my, mirrored mx)
            const float re2 = qr - sr, im2 = qi + si;   // (mirrored my, mx)
            const float re3 = qr + sr, im3 = qi - si;   // (mirrored my, mirrored mx)
            const int i = i4 * 4 + u;
            sum[0][i] = fmaf(w, re0 * re0 + im0 * im0, sum[0][i]);
            sum[1][i] = fmaf(w, re1 * re1 + im1 * im1, sum[1][i]);
            sum[2][i] = fmaf(w, re2 * re2 + im2 * im2, sum[2][i]);
            sum[3][i] = fmaf(w, re3 * re3 + im3 * im3, sum[3][i]);
            if (FIELD) {
              fe[0][FIELD ? u : 0] = make_float2(re0, im0); fe[FIELD ? 1 : 0][FIELD ? u : 0] = make_float2(re1, im1);
              fe[FIELD ? 2 : 0][FIELD ? u : 0] = make_float2(re2, im2); fe[FIELD ? 3 : 0][FIELD ? u : 0] = make_float2(re3, im3);
            }
          }
          if constexpr (FIELD)
            store_field_group(P.field + ((size_t)c * P.Z + (P.z0 + zl)) * (size_t)P.M * P.M, P.M, P.m, ty * 128 + q * 32, lane,
                              tx * 64 + e * 16 + i4 * 4, fe, P.fscale, (P.M & 7) == 0);
        }
      }
      // coalesced store of the four mirrored quadrants through the padded staging tile
      float *Ib = P.intensity + (size_t)(P.z0 + zl) * P.M * P.M;
#pragma unroll
      for (int qd = 0; qd < 4; ++qd) {
        named_bar_sync(1, 32 * K2P_EPI_WARPS);
        float *srow = staging + (q * 32 + lane) * K2P_PITCH + e * 16;
#pragma unroll
        for (int i = 0; i < 16; ++i) srow[i] = sum[qd][i];
        named_bar_sync(1, 32 * K2P_EPI_WARPS);
#pragma unroll
        for (int rr = 0; rr < 8; ++rr) {
          const int row = wi * 8 + rr;
          const int my = ty * 128 + row;
          if (my < P.m) {
            const int y = (qd & 2) ? P.M - 1 - my : my;
#pragma unroll
            for (int h = 0; h < 2; ++h) {
              const int col = h * 32 + lane;
              const int mx = tx * 64 + col;
              if (mx < P.m) {
                const int x = (qd & 1) ? P.M - 1 - mx : mx;
                __stcs(Ib + (size_t)y * P.M + x, staging[row * K2P_PITCH + col]);   // streaming: the output should not displace T^T in L2
              }
            }
          }
        }
      }
    }
  }
}

template <bool FIELD>
__global__ void __cluster_dims__(2, 1, 1) __launch_bounds__(K2P_THREADS, 1)
k2_pair(const __grid_constant__ CUtensorMap map_xhi, const __grid_constant__ CUtensorMap map_xlo,
        const __grid_constant__ CUtensorMap map_thi, const __grid_constant__ CUtensorMap map_tlo, const K2PArgs P) {
  extern __shared__ uint8_t smem_raw[];
  uint8_t *smem = (uint8_t *)(((uintptr_t)smem_raw + 1023) & ~(uintptr_t)1023);
  // (pointer arithmetic on the shared array: the compiler keeps the address space, the epilogue's staging accesses are LDS / STS
  // instead of generic loads and stores)
  float *staging = reinterpret_cast<float *>(smem_raw + ((1024u - (smem_u32(smem_raw) & 1023u)) & 1023u) + K2P_NST * P_STAGE);
  __shared__ K2PShared S;
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const uint32_t rank = cluster_ctarank();

  if (threadIdx.x == 0) {
    for (int i = 0; i < K2P_NST; ++i) { mbar_init(&S.full[i], 1); mbar_init(&S.empty[i], 1); }
    mbar_init(&S.acc_full, 1);
    mbar_init(&S.acc_empty, 2 * K2P_EPI_WARPS);
    fence_barrier_init();
  }
  if (warp == 0 && lane == 0) { prefetch_tmap(&map_xhi); prefetch_tmap(&map_xlo); prefetch_tmap(&map_thi); prefetch_tmap(&map_tlo); }
  if (warp == 1) tmem_alloc2(&S.tmem_slot, 512);
  tcgen05_fence_before();
  __syncthreads();
  cluster_sync_all();                       // the peer's barriers are initialised before anything remote touches them
  tcgen05_fence_after();
  const uint32_t tmem = S.tmem_slot;

  const int nk = P.n_pad / 64;
  const int tiles_yp = (P.m_pad / 128 + 1) / 2, tiles_x = P.m_pad / 64;
  const int ntiles = P.zc * tiles_yp * tiles_x;
  const int ncl = gridDim.x >> 1, cid = blockIdx.x >> 1;

  // register budget: launch = 640 x 96; the four feeder warps drop to 24 registers, the sixteen epilogue warps take 112 (128 x 24 + 512 x 112 <= 640 x 96)
  if (warp < 4) {
    setmaxnreg_dec<24>();
    k2p_feed<false>(smem, S, tmem, map_xhi, map_xlo, map_thi, map_tlo, P, warp, rank, nk, tiles_yp, tiles_x, ntiles, ncl, cid, FuseCtx{});
  } else {
    setmaxnreg_inc<112>();
    k2p_epilogue<FIELD>(staging, S, tmem, P, warp, lane, rank, tiles_yp, tiles_x, ntiles, ncl, cid);
  }
  tcgen05_fence_before();
  __syncthreads();
  cluster_sync_all();
  if (warp == 1) tmem_dealloc2(tmem, 512);
}

// ---- stage 1 ----------------------------------------------------------------------------------------------------------
struct K1PArgs {
  const float4 *bgp;    // [2][C][jt][kc][half][8 samples][256 threads]  base pupil (4 slots), pre-scaled by s_Q
  size_t bgp_plane;     // float4 elements between the tables of consecutive planes: 0 = one static table (the normal case);
                        // > 0 = "materialised pupil": every plane brings its own folded pupil (the adjoint's back-projection)
  const float4 *ktq;    // [jt][kc][half][4 sample pairs][256 threads]      kappa / 2 pi (hi, lo) of two samples
  const float4 *planes; // [Z]
  int C, n_pad, m_pad, z0, zc;
  float f1;             // epilogue factor s_T / (s_Q s_X)
  int handoff;          // how the non-leader CTA's producer warps signal the leader's barrier: 0 plain arrive, 1 cluster-scope release
  int defer;            // K = 16 steps of the next stage issued before a stage buffer is released (0 = released right behind its own stage)
  int waitfirst;        // 1: producers wait for the operand slot before they compute its rows (see k1p_produce)
  int asplit;           // 1: the table half of a stage buffer (refilled by TMA, no hazard) has its own barrier and is released right
                        // behind its own stage; only the producer-written half waits for the deferred release
};

constexpr int K1P_NST = 2;
constexpr int K1P_PRODUCER_WARPS = 8;
constexpr int K1P_FEED_WARPS = 4;                                  // table TMA, MMA, idle, base-pupil copies: roles fill whole warpgroups (setmaxnreg)
constexpr int K1P_THREADS = 32 * (K1P_FEED_WARPS + K1P_PRODUCER_WARPS + 4);
constexpr int K1P_STAGING = 2 * TILE16K;                          // hi tile + lo tile of one chain: 128 mx x 64 qy each
constexpr int K1P_BB_SLOTS = 2;
constexpr int K1P_BB_BYTES = 8 * 256 * 16;                        // one stage of base pupil for this CTA: 8 samples x 256 threads x float4
constexpr int K1P_MAX_NK = 4;                                     // k-chunks whose defocus phasors the producers keep in registers per tile (n_pad <= 256)
constexpr int K1P_SMEM = 1024 + K1P_NST * P_STAGE + K1P_STAGING + K1P_BB_SLOTS * K1P_BB_BYTES;
constexpr int K1P_QY = 64;                                        // q_y per tile (32 generated by each CTA)

struct K1PShared {
  uint64_t full[K1P_NST], empty[K1P_NST], acc_full[2], acc_empty[2];
  uint64_t a_empty[K1P_NST];                                // table half of a stage buffer (asplit)
  uint64_t bb_full[K1P_BB_SLOTS], bb_empty[K1P_BB_SLOTS];   // base-pupil ring: bulk copy -> producers -> free
  uint32_t tmem_slot;
};
struct K1PGeom { int nk, tiles_j, tiles_m, ntiles, ncl, cid, nitems; };

// Two tilings share the kernel (template parameter GM):
//   GM = false (m_pad a multiple of 256): a tile is (plane, 64 q_y, 256 m_x); the CTAs of a pair hold the two 128-row halves
//       of the table rows (A) and generate the two 32-q_y halves of the pupil rows (B); 2 C items (component, x-parity group)
//       per tile, every accumulator column is used.
//   GM = true ("group mode", m_pad an odd multiple of 128, i.e. output half-sizes up to 128 and 257..384, ...): a tile is
//       (plane, 32 q_y, 128 m_x) and the pair splits by x-parity GROUP instead: CTA 0 holds the cos rows of the 128 m_x and
//       generates the x-even chains, CTA 1 holds the sin rows and generates the x-odd chains, C items per tile.  Each CTA's
//       accumulator half that multiplies its table with the other group's chains is computed and discarded: half of the
//       tensor work is waste, in exchange for the pair kernel's producer / epilogue machinery on shapes that have only 128
//       output rows (before: the single-CTA k1_tc at 0.24 of the tensor peak, issue-bound).
template <bool GM> struct K1PTile {
  int mt, jt, zl, jt64, half;
  __device__ __forceinline__ K1PTile(int t, const K1PGeom &G, uint32_t rank) {
    mt = t % G.tiles_m;
    const int r = t / G.tiles_m;
    jt = r % G.tiles_j;
    zl = r / G.tiles_j;
    jt64 = GM ? (jt >> 1) : jt;
    half = GM ? (jt & 1) : (int)rank;            // which 32-q_y half of the 64-q_y table block this CTA generates
  }
};

// 1-D bulk copy global -> shared of this CTA, completion bytes on a local mbarrier
__device__ __forceinline__ void bulk_load_1d(uint32_t smem_dst, const void *gsrc, uint32_t bytes, uint64_t *bar) {
  asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];"
               ::"r"(smem_dst), "l"((uint64_t)gsrc), "r"(bytes), "r"(smem_u32(bar))
               : "memory");
}
__device__ __forceinline__ float4 ld_shared_v4f(uint32_t saddr) {
  float4 v;
  asm volatile("ld.shared.v4.f32 {%0, %1, %2, %3}, [%4];" : "=f"(v.x), "=f"(v.y), "=f"(v.z), "=f"(v.w) : "r"(saddr));
  return v;
}

// TMA warp (both CTAs: table rows of the CTA's own 128 mx) and MMA warp (leader CTA)
template <bool GM>
__device__ __forceinline__ void k1p_feed(uint8_t *smem, K1PShared &S, uint32_t tmem, const CUtensorMap &map_xhi, const CUtensorMap &map_xlo,
                                         const K1PArgs &P, const K1PGeom &G, int warp, uint32_t rank) {
  const bool leader = rank == 0;
  if (warp == 0) {
    if (elect_one()) {
      int st = 0, ph = 0;
      uint32_t full_leader[K1P_NST];
      for (int i = 0; i < K1P_NST; ++i) full_leader[i] = mapa(smem_u32(&S.full[i]), 0);
      for (int t = G.cid; t < G.ntiles; t += G.ncl) {
        const int mt = t % G.tiles_m;
        for (int cg = 0; cg < G.nitems; ++cg) {
          const int row = GM ? (int)rank * P.m_pad + mt * 128 : (cg & 1) * P.m_pad + mt * 256 + (int)rank * 128;
          for (int kc = 0; kc < G.nk; ++kc) {
            mbar_wait(P.asplit ? &S.a_empty[st] : &S.empty[st], ph ^ 1);
            const uint32_t s = smem_u32(smem + st * P_STAGE);
            if (leader) mbar_arrive_expect_tx(&S.full[st], 4 * TILE16K);
            tma2_load_2d(s, &map_xhi, full_leader[st], kc * 64, row);
            tma2_load_2d(s + TILE16K, &map_xlo, full_leader[st], kc * 64, row);
            if (++st == K1P_NST) { st = 0; ph ^= 1; }
          }
        }
      }
    }
  } else if (warp == 1) {
    if (leader && elect_one()) {
      int st = 0, ph = 0, it = 0, pending = -1;
      for (int t = G.cid; t < G.ntiles; t += G.ncl) {
        for (int cg = 0; cg < G.nitems; ++cg, ++it) {
          const int g = it & 1;                                      // accumulator half (= the x-parity group when GM is false)
          mbar_wait(&S.acc_empty[g], ((it >> 1) & 1) ^ 1);
          tcgen05_fence_after();
          const uint32_t d = tmem + g * 256;
          for (int kc = 0; kc < G.nk; ++kc) {
            if (P.handoff == 1) mbar_wait_acquire_cluster(&S.full[st], ph);
            else mbar_wait(&S.full[st], ph);
            tcgen05_fence_after();
            const uint32_t sb = smem_u32(smem + st * P_STAGE);
#pragma unroll
            for (int k = 0; k < 4; ++k) {
              issue_kstep2(sb, d, k, kc == 0 && k == 0);
              // Happens-before chains of an operand slot `st`, edge by edge, and what each edge rests on:
              //  read-after-write (producers -> tensor core):
              //    st.shared of the operand rows (generic proxy)
              //    -> fence.proxy.async.shared::cta in every writing thread (PTX ISA, async proxy: generic-proxy accesses before
              //       the fence are ordered before later async-proxy accesses - the tcgen05.mma operand reads)
              //    -> __syncwarp, lane 0: mbarrier.arrive on the LEADER's `full[st]` (default semantics: .release at .cta scope;
              //       PSF_TUNE_K1P_HANDOFF = 1: .release.cluster)
              //    -> this thread: mbarrier.try_wait (default .acquire.cta; HANDOFF = 1: .acquire.cluster)
              //    -> tcgen05.fence::after_thread_sync -> tcgen05.mma.cta_group::2 (reads the slot in both CTAs).
              //    For the leader's own producers every edge is in the memory model.  For the peer's producers the release /
              //    acquire pair is morally strong only at cluster scope: HANDOFF = 1 is the chain the model guarantees, and it costs
              //    17 % of the stage-1 time (the release compiles to MEMBAR.ALL.GPU + ERRBAR on the stage's critical path).  The
              //    default rests on the hardware order "stores performed -> fence retires -> the remote arrive leaves the SM";
              //    the operand rows of the peer live in the peer's own shared memory and are read by the peer's tensor core.
              //  write-after-read (tensor core -> producers):
              //    tcgen05.mma x 12 -> tcgen05.commit.cta_group::2 ... multicast::cluster on `empty[st]` of both CTAs (PTX ISA: the
              //    arrive is triggered when all prior asynchronous tcgen05 operations of the issuing thread have completed)
              //    -> producer: mbarrier.try_wait -> st.shared into the slot.  Every edge is in the model - and this is where the
              //    measured failures sit (profiles/r5_soak.md: the cluster-scope pair above still fails without the deferral, so
              //    the read-after-write side is not it): hence the margin below, P.defer K-steps (default 2; alone: 1 -> one
              //    wrong stack in 25000 calls, 0 -> one in 100, and 2 failed once in 150000 in one build), and the producers'
              //    wait-first order (P.waitfirst in k1p_produce), which puts their computation between the observed release
              //    and the first store.
              // Deferred release (profiles/r1j_race_k1_pair.md): the commit tracks the UMMAs of the issuing (leader) CTA; in
              // the peer, whose tensor core can trail by a little, producers with their rows ready in registers
              // overwrote the operand tile while it was still being read.  The previous stage's buffer is therefore
              // released only after K1P_DEFER K-steps of this stage have been issued behind it: the commit then also
              // waits for those, which gives the peer that much tensor time of slack.
              if (pending >= 0) {
                // (diagnosis settings HANDOFF = 2 / 3, profiles/r5_soak.md: the slot of one CTA released one K-step late, the other's two)
                const int dl = P.handoff == 2 ? 1 : (P.handoff == 3 ? 2 : P.defer), dp = P.handoff == 2 ? 2 : (P.handoff == 3 ? 1 : P.defer);
                if (dl == dp) {
                  if (k == dl - 1) { umma2_commit(&S.empty[pending]); pending = -1; }
                } else {
                  if (k == dl - 1) umma2_commit(&S.empty[pending], 1);
                  if (k == dp - 1) umma2_commit(&S.empty[pending], 2);
                  if (k == (dl > dp ? dl : dp) - 1) pending = -1;
                }
              }
            }
            if (P.asplit) umma2_commit(&S.a_empty[st]);          // the TMA-written table tiles: free as soon as these UMMAs are done
            if (P.defer == 0) umma2_commit(&S.empty[st]);
            else pending = st;
            if (++st == K1P_NST) { st = 0; ph ^= 1; }
          }
          umma2_commit(&S.acc_full[g]);
        }
      }
      if (pending >= 0) umma2_commit(&S.empty[pending]);
    }
  } else if (warp == 3) {
    // Base-pupil copies: one 32 KB bulk copy per stage (the table is stored in the producers' read order, so a stage
    // of this CTA is one contiguous block) into a two-slot ring.  The producers then only read shared memory: no
    // global-load latency in their loop.
    if (elect_one()) {
      int bs = 0, bph = 0;
      const uint32_t ring = smem_u32(smem + K1P_NST * P_STAGE + K1P_STAGING);
      for (int t = G.cid; t < G.ntiles; t += G.ncl) {
        const K1PTile<GM> T(t, G, rank);
        for (int cg = 0; cg < G.nitems; ++cg) {
          const int grp = GM ? (int)rank : (cg & 1), c = GM ? cg : (cg >> 1);
          const float4 *src = P.bgp + (size_t)(P.z0 + T.zl) * P.bgp_plane + (size_t)(grp * P.C + c) * P.n_pad * P.n_pad;
          for (int kc = 0; kc < G.nk; ++kc) {
            mbar_wait(&S.bb_empty[bs], bph ^ 1);
            mbar_arrive_expect_tx(&S.bb_full[bs], K1P_BB_BYTES);
            bulk_load_1d(ring + bs * K1P_BB_BYTES, src + ((size_t)(T.jt64 * G.nk + kc) * 2 + T.half) * 2048, K1P_BB_BYTES, &S.bb_full[bs]);
            if (++bs == K1P_BB_SLOTS) { bs = 0; bph ^= 1; }
          }
        }
      }
    }
  }
}

// Eight producer warps: this CTA's 32 q_y x 4 slots = 128 B-operand rows per stage; a thread owns 8 consecutive q_x of one
// q_y row.  The defocus phasor of a sample is the same for all 2 C (component, group) items of a tile: the thread
// computes its 8 x nk phasors at the first item and keeps them in registers (the k-chunk loop is unrolled).  The base
// pupil of the stage comes from the shared-memory ring filled by the copy warp.
template <bool GM>
__device__ __forceinline__ void k1p_produce(uint8_t *smem, K1PShared &S, const K1PArgs &P, const K1PGeom &G, int lane, uint32_t rank) {
  const int tid = threadIdx.x - 32 * K1P_FEED_WARPS;
  const int ql = tid >> 3, cgp = tid & 7;                        // row within the CTA's 32 q_y, 16-byte chunk (8 q_x)
  // swizzled byte offset of chunk cgp in row (slot*32 + ql): rows 128 B apart, chunk ^= row & 7
  const uint32_t off0 = (uint32_t)ql * 128u + (((uint32_t)cgp ^ ((uint32_t)ql & 7u)) << 4);
  const uint32_t smem0 = smem_u32(smem);
  const uint32_t full_leader0 = mapa(smem_u32(&S.full[0]), 0);
  const uint32_t ring = smem0 + K1P_NST * P_STAGE + K1P_STAGING + (uint32_t)tid * 16u;   // [slot][sample e][thread] float4
  int st = 0, ph = 0, bs = 0, bph = 0;
  float4 sc[K1P_MAX_NK][4];                                      // (cos, sin) of samples (2i, 2i+1) of k-chunk kc (mod 4)
  const bool cached = G.nk <= K1P_MAX_NK;                        // larger pupils recompute the phasors at every stage
  float4 kt[4];
  // kappa of (tile, kc): [jt][kc][half][4 sample pairs][256 threads] float4
  auto load_kt = [&](int t, int kc) {                           // kappa of (tile t, k-chunk kc)
    const K1PTile<GM> T(t, G, rank);
    const float4 *k4 = P.ktq + ((size_t)(T.jt64 * G.nk + kc) * 2 + T.half) * 1024 + tid;
#pragma unroll
    for (int i = 0; i < 4; ++i) kt[i] = __ldg(k4 + i * 256);
  };
  if (G.cid < G.ntiles) load_kt(G.cid, 0);
  for (int t = G.cid; t < G.ntiles; t += G.ncl) {
    const K1PTile<GM> T(t, G, rank);
    const float4 pl = __ldg(P.planes + P.z0 + T.zl);
    for (int cg = 0; cg < G.nitems; ++cg) {
     for (int kcb = 0; kcb < G.nk; kcb += K1P_MAX_NK) {
#pragma unroll
      for (int k4 = 0; k4 < K1P_MAX_NK; ++k4) {
        const int kc = kcb + k4;
        if (kc < G.nk) {
          if (cg == 0 || !cached) {
#pragma unroll
            for (int i = 0; i < 4; ++i) {
              const float t0 = 6.283185307179586f * kz_turns(make_float2(kt[i].x, kt[i].y), pl.x, pl.y);
              const float t1 = 6.283185307179586f * kz_turns(make_float2(kt[i].z, kt[i].w), pl.x, pl.y);
              sc[k4][i] = make_float4(__cosf(t0), __sinf(t0), __cosf(t1), __sinf(t1));
            }
          }
          // The operand slot is awaited BEFORE the rows are computed (P.waitfirst, default): the producers are the slower side
          // of the pipeline, so the slot is almost always free already and nothing is lost - but when it is not, the math and
          // the split below (about 600 cycles) now lie between the moment the release is observed and the first store into
          // the slot, on top of the deferral of the release itself (profiles/r5_soak.md).
          if (P.waitfirst) mbar_wait(&S.empty[st], ph ^ 1);
          mbar_wait(&S.bb_full[bs], bph);
          uint32_t hi[4][4], lo[4][4];                             // [slot][pair of q_x]
#pragma unroll
          for (int i = 0; i < 4; ++i) {
            const float4 b0 = ld_shared_v4f(ring + bs * K1P_BB_BYTES + (2 * i) * 4096);
            const float4 b1 = ld_shared_v4f(ring + bs * K1P_BB_BYTES + (2 * i + 1) * 4096);
            const float cs0 = sc[k4][i].x, sn0 = sc[k4][i].y, cs1 = sc[k4][i].z, sn1 = sc[k4][i].w;
            split_f16x2(b0.x * cs0 - b0.y * sn0, b1.x * cs1 - b1.y * sn1, hi[0][i], lo[0][i]);
            split_f16x2(b0.x * sn0 + b0.y * cs0, b1.x * sn1 + b1.y * cs1, hi[1][i], lo[1][i]);
            split_f16x2(b0.z * cs0 - b0.w * sn0, b1.z * cs1 - b1.w * sn1, hi[2][i], lo[2][i]);
            split_f16x2(b0.z * sn0 + b0.w * cs0, b1.z * sn1 + b1.w * cs1, hi[3][i], lo[3][i]);
          }
          __syncwarp();
          if (lane == 0) mbar_arrive(&S.bb_empty[bs]);             // the ring slot is in registers
          if (++bs == K1P_BB_SLOTS) { bs = 0; bph ^= 1; }
          if (!P.waitfirst) mbar_wait(&S.empty[st], ph ^ 1);
          const uint32_t bh = smem0 + st * P_STAGE + 2 * TILE16K + off0, bl = bh + TILE16K;
#pragma unroll
          for (int s = 0; s < 4; ++s) {
            st_shared_v4(bh + s * 4096, hi[s][0], hi[s][1], hi[s][2], hi[s][3]);
            st_shared_v4(bl + s * 4096, lo[s][0], lo[s][1], lo[s][2], lo[s][3]);
          }
          fence_proxy_async_smem();                                // every writer fences its own stores; no load is in flight here
          __syncwarp();
          if (lane == 0) {
            if (rank == 0 || P.handoff != 1) mbar_arrive_cluster(full_leader0 + st * 8);
            else mbar_arrive_cluster_release(full_leader0 + st * 8);
          }
          if (++st == K1P_NST) { st = 0; ph ^= 1; }
          // kappa of the stage that computes phasors next (one stage ahead), issued after the fence so that the fence's
          // memory barrier never waits for it
          if (cached) {
            if (cg == 0 && kc + 1 < G.nk) load_kt(t, kc + 1);
            if (cg == G.nitems - 1 && kc == G.nk - 1 && t + G.ncl < G.ntiles) load_kt(t + G.ncl, 0);
          } else if (kc + 1 < G.nk) {
            load_kt(t, kc + 1);
          } else if (cg + 1 < G.nitems) {
            load_kt(t, 0);
          } else if (t + G.ncl < G.ntiles) {
            load_kt(t + G.ncl, 0);
          }
        }
      }
     }
    }
  }
}

// Four epilogue warps: TMEM -> scale -> fp16 hi / lo -> swizzled staging tiles -> TMA store of T^T[chain][mx][qy].
// The hi tile and the lo tile are separate buffers, each stored by its own bulk group, so writing one overlaps the
// TMA read of the other.  GM = false: 64 q_y per row (128-byte rows, SWIZZLE_128B); GM = true: this CTA's own 128
// accumulator columns only, 32 q_y per row (64-byte rows, SWIZZLE_64B: 16-byte chunk ^= (row >> 1) & 3).
template <bool GM, bool FUSED>
__device__ __forceinline__ void k1p_epilogue(uint8_t *smem, K1PShared &S, uint32_t tmem, const CUtensorMap &map_this, const CUtensorMap &map_tlos,
                                             const K1PArgs &P, const K1PGeom &G, int warp, int lane, uint32_t rank, const FuseCtx &F) {
  const int q = warp & 3;                       // TMEM lane quarter = 32 of this CTA's 128 mx rows
  const int row = q * 32 + lane;
  const int et = threadIdx.x - 32 * (K1P_FEED_WARPS + K1P_PRODUCER_WARPS);   // 0..127
  const uint32_t stg0 = smem_u32(smem + K1P_NST * P_STAGE);
  const uint32_t stg_hi = stg0 + (uint32_t)row * (GM ? 64u : 128u), stg_lo = stg_hi + TILE16K;
  const uint32_t acc_empty_leader = mapa(smem_u32(&S.acc_empty[0]), 0);
  const uint32_t swz = GM ? (((uint32_t)row >> 1) & 3u) : ((uint32_t)row & 7u);
  int it = 0;
  for (int t = G.cid; t < G.ntiles; t += G.ncl) {
    const K1PTile<GM> T(t, G, rank);
    const int mx0 = GM ? T.mt * 128 : T.mt * 256 + (int)rank * 128;
    const int qy0 = T.jt * (GM ? 32 : K1P_QY);
    for (int cg = 0; cg < G.nitems; ++cg, ++it) {
      const int g = it & 1;                                            // accumulator half
      const int grp = GM ? (int)rank : (cg & 1), c = GM ? cg : (cg >> 1);
      int unit = T.zl * P.C + c;
      if (FUSED) {
        const FuseUnit fu = fuse_unit(F, P.C, T.zl, c);
        unit = fu.ring;
        // first item of a component: its ring slot must have been read by every stage-2 cluster of the unit before it
        if (et == 0 && grp == 0 && fu.prev >= 0) fuse_wait(F, F.consumed + fu.prev, F.a2);
      }
      mbar_wait(&S.acc_full[g], (it >> 1) & 1);
      tcgen05_fence_after();
#pragma unroll 1
      for (int s = 0; s < (GM ? 2 : 4); ++s) {
        // GM false: round s = slot s (one chain), both q_y halves.  GM true: round s = slots 2 s and 2 s + 1 of this CTA's
        // group = two consecutive chains, stored by one TMA box of 2 chains (the staging tile holds them back to back).
        const int chain = unit * 8 + (GM ? s * 4 + grp * 2 : (s >> 1) * 4 + grp * 2 + (s & 1));
        uint32_t pl[2][16];
        // the hi buffer was handed to the TMA store two bulk groups ago (hi, lo of the previous slot)
        if (et == 0) bulk_wait_read<1>();
        named_bar_sync(2, 128);
#pragma unroll
        for (int h = 0; h < 2; ++h) {            // GM false: q_y half h was generated by CTA h: columns h*128 + s*32 + 0..31
          uint32_t v[32], ph[16];
          tmem_ld_32x32b_x32(tmem + ((uint32_t)(q * 32) << 16) + g * 256 + (GM ? (int)rank * 128 + (2 * s + h) * 32 : h * 128 + s * 32), v);
          tmem_ld_wait();
#pragma unroll
          for (int e = 0; e < 16; ++e)
            split_f16x2(__uint_as_float(v[2 * e]) * P.f1, __uint_as_float(v[2 * e + 1]) * P.f1, ph[e], pl[h][e]);
#pragma unroll
          for (int j = 0; j < 4; ++j)            // GM false: 16-byte chunk h*4 + j of the 128-byte row; GM true: chunk j of the 64-byte row of chain h
            st_shared_v4(stg_hi + (GM ? (uint32_t)h * 8192u + ((((uint32_t)j) ^ swz) << 4) : ((((uint32_t)(h * 4 + j)) ^ swz) << 4)),
                         ph[4 * j], ph[4 * j + 1], ph[4 * j + 2], ph[4 * j + 3]);
        }
        if (s == (GM ? 1 : 3)) {                 // every TMEM read of this item is done: release the accumulator
          tcgen05_fence_before();
          __syncwarp();
          if (lane == 0) mbar_arrive_cluster(acc_empty_leader + g * 8);
        }
        fence_proxy_async_smem();
        named_bar_sync(2, 128);
        if (et == 0) {
          tma_store_3d(&map_this, stg0, qy0, mx0, chain);
          bulk_commit();
          bulk_wait_read<1>();                   // the lo buffer of the previous slot has been read
        }
        named_bar_sync(2, 128);
#pragma unroll
        for (int h = 0; h < 2; ++h)
#pragma unroll
          for (int j = 0; j < 4; ++j)
            st_shared_v4(stg_lo + (GM ? (uint32_t)h * 8192u + ((((uint32_t)j) ^ swz) << 4) : ((((uint32_t)(h * 4 + j)) ^ swz) << 4)),
                         pl[h][4 * j], pl[h][4 * j + 1], pl[h][4 * j + 2], pl[h][4 * j + 3]);
        fence_proxy_async_smem();
        named_bar_sync(2, 128);
        if (et == 0) {
          tma_store_3d(&map_tlos, stg0 + TILE16K, qy0, mx0, chain);
          bulk_commit();
        }
      }
      if (FUSED && et == 0 && cg >= 1) {
        // an item issues 8 bulk groups (4 slots x hi, lo): everything older than the last 8 has completed, i.e. item cg - 1
        bulk_wait_complete<8>();
        if ((cg - 1) & 1) {                      // item cg - 1 was the second (last) item of component (cg - 1) / 2
          fence_proxy_async_all();
          red_release_gpu_add(F.ready + T.zl * P.C + ((cg - 1) >> 1), 1);
        }
      }
    }
    if (FUSED && et == 0) {                      // last component of the tile
      bulk_wait_complete<0>();
      fence_proxy_async_all();
      red_release_gpu_add(F.ready + T.zl * P.C + (P.C - 1), 1);
    }
  }
  if (et == 0) bulk_wait_all();
}

template <bool GM>
__global__ void __cluster_dims__(2, 1, 1) __launch_bounds__(K1P_THREADS, 1)
k1_pair(const __grid_constant__ CUtensorMap map_xhi, const __grid_constant__ CUtensorMap map_xlo,
        const __grid_constant__ CUtensorMap map_this, const __grid_constant__ CUtensorMap map_tlos, const K1PArgs P) {
  extern __shared__ uint8_t smem_raw[];
  uint8_t *smem = (uint8_t *)(((uintptr_t)smem_raw + 1023) & ~(uintptr_t)1023);
  __shared__ K1PShared S;
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const uint32_t rank = cluster_ctarank();
  if (threadIdx.x == 0) tc::pdl_trigger();                 // the stage-2 grid may take the SMs this grid leaves (it waits for our completion)

  if (threadIdx.x == 0) {
    for (int i = 0; i < K1P_NST; ++i) {
      mbar_init(&S.full[i], 1 + 2 * K1P_PRODUCER_WARPS);  // the leader's expect_tx arrive + every producer warp of the pair
      mbar_init(&S.empty[i], 1);
      mbar_init(&S.a_empty[i], 1);
    }
    for (int i = 0; i < K1P_BB_SLOTS; ++i) { mbar_init(&S.bb_full[i], 1); mbar_init(&S.bb_empty[i], K1P_PRODUCER_WARPS); }
    for (int i = 0; i < 2; ++i) { mbar_init(&S.acc_full[i], 1); mbar_init(&S.acc_empty[i], 8); }
    fence_barrier_init();
  }
  if (warp == 0 && lane == 0) { prefetch_tmap(&map_xhi); prefetch_tmap(&map_xlo); prefetch_tmap(&map_this); prefetch_tmap(&map_tlos); }
  if (warp == 1) tmem_alloc2(&S.tmem_slot, 512);
  tcgen05_fence_before();
  __syncthreads();
  cluster_sync_all();
  tcgen05_fence_after();
  const uint32_t tmem = S.tmem_slot;

  K1PGeom G;
  G.nk = P.n_pad / 64;
  G.tiles_j = P.n_pad / (GM ? 32 : K1P_QY);
  G.tiles_m = P.m_pad / (GM ? 128 : 256);
  G.ntiles = P.zc * G.tiles_j * G.tiles_m;                        // a tile = (plane, q_y tile, m_x tile); the items loop inside
  G.nitems = GM ? P.C : 2 * P.C;
  G.ncl = gridDim.x >> 1;
  G.cid = blockIdx.x >> 1;

  // register budget (launch: 512 x 128; setmaxnreg acts on whole warpgroups): feeders 24, producers 184, epilogue 104
  if (warp < K1P_FEED_WARPS) {
    setmaxnreg_dec<24>();
    k1p_feed<GM>(smem, S, tmem, map_xhi, map_xlo, P, G, warp, rank);
  } else if (warp < K1P_FEED_WARPS + K1P_PRODUCER_WARPS) {
    setmaxnreg_inc<184>();
    k1p_produce<GM>(smem, S, P, G, lane, rank);
  } else {
    setmaxnreg_dec<104>();
    k1p_epilogue<GM, false>(smem, S, tmem, map_this, map_tlos, P, G, warp, lane, rank, FuseCtx{});
  }
  tcgen05_fence_before();
  __syncthreads();
  cluster_sync_all();
  if (warp == 1) tmem_dealloc2(tmem, 512);
}

// Both stages in one launch: clusters [0, n1) run the stage-1 roles of k1_pair, the others the stage-2 roles of k2_pair,
// coupled by the flags of FuseCtx.  640 threads as k2_pair; in a stage-1 cluster the fifth warpgroup gives its registers
// back and idles.  Register budget after setmaxnreg (pool 640 x 96): stage 1 24 / 160 / 104 / 24, stage 2 24 / 112.
constexpr int K12_SMEM = K1P_SMEM > K2P_SMEM ? K1P_SMEM : K2P_SMEM;

template <bool FIELD>
__global__ void __cluster_dims__(2, 1, 1) __launch_bounds__(K2P_THREADS, 1)
k12_fused(const __grid_constant__ CUtensorMap map_xhi, const __grid_constant__ CUtensorMap map_xlo,
          const __grid_constant__ CUtensorMap map_this, const __grid_constant__ CUtensorMap map_tlos,
          const __grid_constant__ CUtensorMap map_thi, const __grid_constant__ CUtensorMap map_tlo,
          const K1PArgs P1, const K2PArgs P2, const FuseCtx F) {
  extern __shared__ uint8_t smem_raw[];
  uint8_t *smem = (uint8_t *)(((uintptr_t)smem_raw + 1023) & ~(uintptr_t)1023);
  __shared__ K1PShared S1;
  __shared__ K2PShared S2;
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const uint32_t rank = cluster_ctarank();
  const int cluster = blockIdx.x >> 1, nclusters = gridDim.x >> 1;
  const bool stage1 = cluster < F.n1;

  if (threadIdx.x == 0) {
    if (stage1) {
      for (int i = 0; i < K1P_NST; ++i) { mbar_init(&S1.full[i], 1 + 2 * K1P_PRODUCER_WARPS); mbar_init(&S1.empty[i], 1); mbar_init(&S1.a_empty[i], 1); }
      for (int i = 0; i < K1P_BB_SLOTS; ++i) { mbar_init(&S1.bb_full[i], 1); mbar_init(&S1.bb_empty[i], K1P_PRODUCER_WARPS); }
      for (int i = 0; i < 2; ++i) { mbar_init(&S1.acc_full[i], 1); mbar_init(&S1.acc_empty[i], 8); }
    } else {
      for (int i = 0; i < K2P_NST; ++i) { mbar_init(&S2.full[i], 1); mbar_init(&S2.empty[i], 1); }
      mbar_init(&S2.acc_full, 1);
      mbar_init(&S2.acc_empty, 2 * K2P_EPI_WARPS);
    }
    fence_barrier_init();
  }
  if (warp == 0 && lane == 0) {
    prefetch_tmap(&map_xhi); prefetch_tmap(&map_xlo);
    if (stage1) { prefetch_tmap(&map_this); prefetch_tmap(&map_tlos); } else { prefetch_tmap(&map_thi); prefetch_tmap(&map_tlo); }
  }
  if (warp == 1) tmem_alloc2(stage1 ? &S1.tmem_slot : &S2.tmem_slot, 512);
  tcgen05_fence_before();
  __syncthreads();
  cluster_sync_all();
  tcgen05_fence_after();
  const uint32_t tmem = stage1 ? S1.tmem_slot : S2.tmem_slot;

  if (stage1) {
    K1PGeom G;
    G.nk = P1.n_pad / 64;
    G.tiles_j = P1.n_pad / K1P_QY;
    G.tiles_m = P1.m_pad / 256;
    G.ntiles = P1.zc * G.tiles_j * G.tiles_m;
    G.nitems = 2 * P1.C;
    G.ncl = F.n1;
    G.cid = cluster;
    if (warp < K1P_FEED_WARPS) {
      setmaxnreg_dec<24>();
      k1p_feed<false>(smem, S1, tmem, map_xhi, map_xlo, P1, G, warp, rank);
    } else if (warp < K1P_FEED_WARPS + K1P_PRODUCER_WARPS) {
      setmaxnreg_inc<160>();
      k1p_produce<false>(smem, S1, P1, G, lane, rank);
    } else if (warp < K1P_FEED_WARPS + K1P_PRODUCER_WARPS + 4) {
      setmaxnreg_inc<104>();
      k1p_epilogue<false, true>(smem, S1, tmem, map_this, map_tlos, P1, G, warp, lane, rank, F);
    } else {
      setmaxnreg_dec<24>();
    }
  } else {
    float *staging = reinterpret_cast<float *>(smem_raw + ((1024u - (smem_u32(smem_raw) & 1023u)) & 1023u) + K2P_NST * P_STAGE);   // (shared address space kept)
    const int nk = P2.n_pad / 64;
    const int tiles_yp = (P2.m_pad / 128 + 1) / 2, tiles_x = P2.m_pad / 64;
    const int ntiles = P2.zc * tiles_yp * tiles_x;
    const int ncl = nclusters - F.n1, cid = cluster - F.n1;
    if (warp < 4) {
      setmaxnreg_dec<24>();
      k2p_feed<true>(smem, S2, tmem, map_xhi, map_xlo, map_thi, map_tlo, P2, warp, rank, nk, tiles_yp, tiles_x, ntiles, ncl, cid, F);
    } else {
      setmaxnreg_inc<112>();
      k2p_epilogue<FIELD>(staging, S2, tmem, P2, warp, lane, rank, tiles_yp, tiles_x, ntiles, ncl, cid);
    }
  }
  tcgen05_fence_before();
  __syncthreads();
  cluster_sync_all();
  if (warp == 1) tmem_dealloc2(tmem, 512);
}

}  // namespace pair
}  // namespace psf
