// umma_common.cuh — PTX wrappers (mbarrier, bulk async copy, tcgen05 MMA / TMEM load,
// shared-memory operand and instruction descriptors) and the dynamic tile schedule shared by
// the bf16 and e4m3 expert kernels (expert_umma.cu, expert_fp8.cu).  sm_100a only.
#pragma once
#include <cuda.h>

#include "caee_internal.cuh"

namespace caee_umma {

constexpr int kTileRows = 128;          // UMMA M
constexpr int kATileBytes = 16 * 1024;  // one 128-row weight tile of a stage (64 k bf16 or 128 k e4m3)
constexpr int kAStageBytes = 2 * kATileBytes;  // two tiles per stage: ONE contiguous 32 KB bulk copy
constexpr int kTmemCols = 512;
constexpr int kMaxStages = 8;

// ------------------------------------------------------------------ PTX wrappers
__device__ __forceinline__ uint32_t smem_u32(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }

__device__ __forceinline__ void mbar_init(uint32_t bar, uint32_t count) {
  asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(bar), "r"(count));
}
__device__ __forceinline__ void mbar_arrive(uint32_t bar) {
  asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(bar) : "memory");
}
__device__ __forceinline__ void mbar_arrive_expect_tx(uint32_t bar, uint32_t bytes) {
  asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(bar), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_wait(uint32_t bar, uint32_t parity) {
  asm volatile(
      "{\n\t.reg .pred p;\n\t"
      "WAIT_%=:\n\t"
      "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n\t"
      "@p bra DONE_%=;\n\t"
      "bra WAIT_%=;\n\t"
      "DONE_%=:\n\t}" ::"r"(bar), "r"(parity) : "memory");
}
__device__ __forceinline__ void bulk_g2s(uint32_t dst, const void* src, uint32_t bytes, uint32_t bar) {
  asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(dst),
               "l"(src), "r"(bytes), "r"(bar)
               : "memory");
}
// Expert weights are read exactly once per step and a step streams far more of them than the L2
// holds: fetched with an evict-first policy they pass through the L2 without displacing what the
// rest of the step re-reads every time (router weights, logits, work lists, h, the kernels' code).
__device__ __forceinline__ uint64_t l2_evict_first_policy() {
  uint64_t pol;
  asm volatile("createpolicy.fractional.L2::evict_first.b64 %0, 1.0;" : "=l"(pol));
  return pol;
}
__device__ __forceinline__ void bulk_g2s_stream(uint32_t dst, const void* src, uint32_t bytes, uint32_t bar, uint64_t pol) {
  asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes.L2::cache_hint [%0], [%1], %2, [%3], %4;" ::"r"(dst),
               "l"(src), "r"(bytes), "r"(bar), "l"(pol)
               : "memory");
}
__device__ __forceinline__ void fence_proxy_async_smem() { asm volatile("fence.proxy.async.shared::cta;" ::: "memory"); }
__device__ __forceinline__ void tc_fence_before() { asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory"); }
__device__ __forceinline__ void tc_fence_after() { asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory"); }
__device__ __forceinline__ void tc_commit(uint32_t bar) {
  asm volatile("tcgen05.commit.cta_group::1.mbarrier::arrive::one.shared::cluster.b64 [%0];" ::"r"(bar) : "memory");
}
// D[tmem] (+)= A[smem] * B[smem]^T, kind::f16 (bf16 inputs, fp32 accumulate), M=128, K=16
__device__ __forceinline__ void umma_bf16(uint32_t d_tmem, uint64_t a_desc, uint64_t b_desc, uint32_t idesc, uint32_t acc) {
  asm volatile(
      "{\n\t.reg .pred p;\n\t"
      "setp.ne.b32 p, %4, 0;\n\t"
      "tcgen05.mma.cta_group::1.kind::f16 [%0], %1, %2, %3, p;\n\t}" ::"r"(d_tmem),
      "l"(a_desc), "l"(b_desc), "r"(idesc), "r"(acc)
      : "memory");
}
template <bool kAcc>
__device__ __forceinline__ void umma_bf16_imm(uint32_t d_tmem, uint64_t a_desc, uint64_t b_desc, uint32_t idesc) {
  asm volatile(
      "{\n\t.reg .pred p;\n\t"
      "setp.ne.b32 p, %4, 0;\n\t"
      "tcgen05.mma.cta_group::1.kind::f16 [%0], %1, %2, %3, p;\n\t}" ::"r"(d_tmem),
      "l"(a_desc), "l"(b_desc), "r"(idesc), "n"(kAcc ? 1 : 0)
      : "memory");
}
// D[tmem] (+)= A[smem] * B[smem]^T, kind::f8f6f4 (e4m3 x e4m3, fp32 accumulate), M=128, K=32
template <bool kAcc>
__device__ __forceinline__ void umma_f8_imm(uint32_t d_tmem, uint64_t a_desc, uint64_t b_desc, uint32_t idesc) {
  asm volatile(
      "{\n\t.reg .pred p;\n\t"
      "setp.ne.b32 p, %4, 0;\n\t"
      "tcgen05.mma.cta_group::1.kind::f8f6f4 [%0], %1, %2, %3, p;\n\t}" ::"r"(d_tmem),
      "l"(a_desc), "l"(b_desc), "r"(idesc), "n"(kAcc ? 1 : 0)
      : "memory");
}
__device__ __forceinline__ void umma_f8(uint32_t d_tmem, uint64_t a_desc, uint64_t b_desc, uint32_t idesc, uint32_t acc) {
  asm volatile(
      "{\n\t.reg .pred p;\n\t"
      "setp.ne.b32 p, %4, 0;\n\t"
      "tcgen05.mma.cta_group::1.kind::f8f6f4 [%0], %1, %2, %3, p;\n\t}" ::"r"(d_tmem),
      "l"(a_desc), "l"(b_desc), "r"(idesc), "r"(acc)
      : "memory");
}
// ---- CTA-pair (cta_group::2) variants: the leader CTA (cluster rank 0) issues one MMA of M = 256 whose
// A rows 0-127 / 128-255 and B rows [0, N/2) / [N/2, N) come from the same shared-memory offsets of
// the two CTAs; each CTA's TMEM receives its own 128 rows of D.
__device__ __forceinline__ uint32_t cluster_ctarank() {
  uint32_t r;
  asm volatile("mov.u32 %0, %%cluster_ctarank;" : "=r"(r));
  return r;
}
__device__ __forceinline__ void cluster_sync_all() {
  asm volatile("barrier.cluster.arrive.release.aligned;\n\tbarrier.cluster.wait.acquire.aligned;" ::: "memory");
}
// arrive on the barrier at the same shared-memory offset in CTA `cta` of the cluster
__device__ __forceinline__ void mbar_arrive_remote(uint32_t bar, uint32_t cta) {
  asm volatile(
      "{\n\t.reg .b32 ra;\n\t"
      "mapa.shared::cluster.u32 ra, %0, %1;\n\t"
      "mbarrier.arrive.shared::cluster.b64 _, [ra];\n\t}" ::"r"(bar), "r"(cta)
      : "memory");
}
// wait on a local barrier whose arrivals come from the peer CTA (cluster-scope acquire)
__device__ __forceinline__ void mbar_wait_cluster(uint32_t bar, uint32_t parity) {
  asm volatile(
      "{\n\t.reg .pred p;\n\t"
      "WAITC_%=:\n\t"
      "mbarrier.try_wait.parity.acquire.cluster.shared::cta.b64 p, [%0], %1;\n\t"
      "@p bra DONEC_%=;\n\t"
      "bra WAITC_%=;\n\t"
      "DONEC_%=:\n\t}" ::"r"(bar), "r"(parity) : "memory");
}
template <bool kAcc>
__device__ __forceinline__ void umma_f16_pair_imm(uint32_t d_tmem, uint64_t a_desc, uint64_t b_desc, uint32_t idesc) {
  asm volatile(
      "{\n\t.reg .pred p;\n\t"
      "setp.ne.b32 p, %4, 0;\n\t"
      "tcgen05.mma.cta_group::2.kind::f16 [%0], %1, %2, %3, p;\n\t}" ::"r"(d_tmem),
      "l"(a_desc), "l"(b_desc), "r"(idesc), "n"(kAcc ? 1 : 0)
      : "memory");
}
// completion of the issuing thread's MMAs -> arrive on the barrier at this offset in BOTH CTAs
__device__ __forceinline__ void tc_commit_pair(uint32_t bar) {
  asm volatile("tcgen05.commit.cta_group::2.mbarrier::arrive::one.shared::cluster.multicast::cluster.b64 [%0], %1;" ::"r"(bar),
               "h"((uint16_t)3)
               : "memory");
}

// Programmatic dependent launch: a kernel launched with cudaLaunchAttributeProgrammaticStreamSerialization
// may start while its predecessor in the stream still runs; griddep_wait() returns once the
// predecessor grid has completed and its writes are visible (at once if launched normally);
// griddep_launch() lets the successor's CTAs be scheduled from now on.
__device__ __forceinline__ void griddep_wait() { asm volatile("griddepcontrol.wait;" ::: "memory"); }
__device__ __forceinline__ void griddep_launch() { asm volatile("griddepcontrol.launch_dependents;" ::: "memory"); }

// One lane of a converged warp (the warp must be converged: "elect.sync").  Code around it
// stays warp-uniform, so descriptor arithmetic runs on the uniform datapath instead of being
// moved lane-register -> uniform-register in front of every tcgen05 instruction.
__device__ __forceinline__ bool elect_one() {
  uint32_t pred;
  asm volatile(
      "{\n\t.reg .pred p;\n\t"
      "elect.sync _|p, 0xffffffff;\n\t"
      "selp.u32 %0, 1, 0, p;\n\t}"
      : "=r"(pred));
  return pred != 0;
}
__device__ __forceinline__ void tmem_ld8(uint32_t taddr, uint32_t (&v)[8]) {
  asm volatile("tcgen05.ld.sync.aligned.32x32b.x8.b32 {%0,%1,%2,%3,%4,%5,%6,%7}, [%8];"
               : "=r"(v[0]), "=r"(v[1]), "=r"(v[2]), "=r"(v[3]), "=r"(v[4]), "=r"(v[5]), "=r"(v[6]), "=r"(v[7])
               : "r"(taddr));
}
__device__ __forceinline__ void tmem_ld16(uint32_t taddr, uint32_t (&v)[16]) {
  asm volatile(
      "tcgen05.ld.sync.aligned.32x32b.x16.b32 {%0,%1,%2,%3,%4,%5,%6,%7,%8,%9,%10,%11,%12,%13,%14,%15}, [%16];"
      : "=r"(v[0]), "=r"(v[1]), "=r"(v[2]), "=r"(v[3]), "=r"(v[4]), "=r"(v[5]), "=r"(v[6]), "=r"(v[7]), "=r"(v[8]),
        "=r"(v[9]), "=r"(v[10]), "=r"(v[11]), "=r"(v[12]), "=r"(v[13]), "=r"(v[14]), "=r"(v[15])
      : "r"(taddr));
}
__device__ __forceinline__ void tmem_ld_wait() { asm volatile("tcgen05.wait::ld.sync.aligned;" ::: "memory"); }

// K-major, no-swizzle shared-memory operand descriptor: start address, LBO (k-adjacent core
// matrices) = 128 B, SBO (adjacent 8-row groups) = 1024 B, descriptor version 1 (sm_100).
__device__ __forceinline__ uint64_t make_desc(uint32_t saddr) {
  return (uint64_t)((saddr >> 4) & 0x3FFF) | ((uint64_t)(128 >> 4) << 16) | ((uint64_t)(1024 >> 4) << 32) | (1ull << 46);
}
// kind::f16 instruction descriptor: D fp32, A/B bf16 (format 1) or fp16 (format 0), both K-major,
// M = 128, N = n.
__device__ __forceinline__ uint32_t make_idesc(int n, bool bf16) {
  return (1u << 4) | (bf16 ? ((1u << 7) | (1u << 10)) : 0u) | ((uint32_t)(n >> 3) << 17) |
         ((uint32_t)(kTileRows >> 4) << 24);
}
constexpr int kOobRow = 0x40000000;   // beyond any tensor: the TMA unit writes zeros (padding rows)

// Four rows of 128 bytes (k bytes [col, col + 128) of rows r0..r3) -> 512 bytes at dst, swizzled
__device__ __forceinline__ void tma_gather4(uint32_t dst, const CUtensorMap* tm, uint32_t bar, int col, int r0, int r1, int r2,
                                            int r3) {
  asm volatile(
      "cp.async.bulk.tensor.2d.shared::cluster.global.tile::gather4.mbarrier::complete_tx::bytes [%0], [%1, {%3, %4, %5, %6, %7}], [%2];"
      ::"r"(dst), "l"(tm), "r"(bar), "r"(col), "r"(r0), "r"(r1), "r"(r2), "r"(r3)
      : "memory");
}
// K-major operand descriptor for the 128-byte-swizzled token operand: 8-row atoms of 1024 B (SBO),
// layout type 2 (SWIZZLE_128B), descriptor version 1; a 32-byte k-step advances the start address.
__device__ __forceinline__ uint64_t make_desc_sw128(uint32_t saddr) {
  return (uint64_t)((saddr >> 4) & 0x3FFF) | (1ull << 16) | ((uint64_t)(1024 >> 4) << 32) | (1ull << 46) | (2ull << 61);
}

__device__ __forceinline__ int ld_acquire(const int* p) {
  int v;
  asm volatile("ld.acquire.gpu.global.s32 %0, [%1];" : "=r"(v) : "l"(p) : "memory");
  return v;
}
struct Tile {
  int phase, run, sub;  // sub = ft (phase 1) or op (phase 2)
  int kq;               // phase 1 with a split k range (see KSplit): which quarter of k this sub-tile contracts
};
// Steps of a few tokens have fewer phase-1 tiles than it takes to balance 148 SMs whose shares of the
// HBM bandwidth differ by +-25% (a C4 step of one token: 144 tiles of 1.8 MB, one per SM, the slowest
// SM 48 us against the fastest's 27).  Such steps split every phase-1 tile's k range into `ks` sub-tiles
// (tickets (run, ft, kq), kq fastest).  A sub-tile's epilogue only leaves its partial gate / up sums in
// `part` and counts itself in `cnt`; the tile is FINISHED by a reducer warp (the CTAs' otherwise idle
// warp 3; tiles handed out by a second ticket counter): it waits for the tile's ks partials, adds them
// in ascending kq — a fixed order —, applies SwiGLU, writes h and counts the tile in the run's "h
// complete" counter.  Sub-tiles never wait and all of them hold lower tickets than any phase-2 tile,
// so a reducer's wait and the phase-2 wait on a run's h always end.
struct KSplit {
  float* part;     // [tile_cap][ks][2][kKSplitCols][128] partial sums, tile = (run - run_begin) * P1 + ft
  int32_t* cnt;    // [tile_cap] finished sub-tiles of a tile; reset by the tile's reducer
  int ks;          // 1: never split
  int tile_cap;    // split only while n_runs * P1 <= tile_cap
  int rticket;     // index in wl.sched of the reducers' ticket counter of this launch
};
constexpr int kKSplit = 4;           // sub-tiles per phase-1 tile when a step is split
constexpr int kKSplitCols = 8;       // most tokens of a run in a split step (host: T <= kKSplitCols)
// Host: the split a T-token step may use (kb1 = k stages of a whole phase-1 tile)
inline KSplit caee_ksplit_for(const caee_ctx* c, int T, int kb1, int ticket) {
  const bool on = c->ks_part && c->ks_tile_cap > 0 && T <= kKSplitCols && kb1 % kKSplit == 0;
  return KSplit{c->ks_part, c->ks_cnt, on ? kKSplit : 1, c->ks_tile_cap, c->wl.n_tickets / 2 + ticket};
}
inline size_t caee_ksplit_part_floats(int tile_cap) { return (size_t)tile_cap * kKSplit * 2 * kKSplitCols * kTileRows; }
struct TileMap {
  int n_runs, run_begin, P1, P2;
  int KS = 1;
  __device__ __forceinline__ bool at(int i, Tile& t) const {
    const int t1 = n_runs * P1 * KS;
    t.kq = 0;
    if (i < t1) {
      const int per = P1 * KS, r = i / per, rem = i - r * per;
      t.phase = 1; t.sub = rem / KS; t.kq = rem - t.sub * KS; t.run = run_begin + r;
      return true;
    }
    i -= t1;
    if (i < n_runs * P2) { const int r = i / P2; t.phase = 2; t.sub = i - r * P2; t.run = run_begin + r; return true; }
    return false;
  }
};

// ------------------------------------------------------------------ the kernel
constexpr int kQueue = 4;      // tile-queue depth (producer runs at most this many tiles ahead)
constexpr int kLag = 3;        // token-operand stages each loader warp keeps in flight (cp.async groups), < ring depth

// Next tile index for a role.  The weight producer claims tiles with one atomic ticket per
// tile and broadcasts them through a small shared-memory queue; every other role pops the
// same sequence.  Tickets are claimed in increasing order, phase-1 tiles have the lower
// tickets, and a phase-1 tile never waits on another tile: a phase-2 tile's wait for its
// run's h therefore always ends (the CTAs holding those phase-1 tickets are running).
struct TileQueue {
  uint32_t full0, empty0;  // mbarrier addresses
  int* slots;
  int q, ph;
  __device__ __forceinline__ int pop() {
    mbar_wait(full0 + 8 * q, ph);
    const int t = slots[q];
    __syncwarp();
    if ((threadIdx.x & 31) == 0) mbar_arrive(empty0 + 8 * q);
    if (++q == kQueue) { q = 0; ph ^= 1; }
    return t;
  }
  // the same for a role that runs on a single lane
  __device__ __forceinline__ int pop1() {
    mbar_wait(full0 + 8 * q, ph);
    const int t = slots[q];
    mbar_arrive(empty0 + 8 * q);
    if (++q == kQueue) { q = 0; ph ^= 1; }
    return t;
  }
};


// Host: 2D byte tensor map over a [rows, row_bytes] array for tile::gather4 row gathers of 128-byte
// pieces with the 128-byte swizzle (box = {128 bytes, 1 row}).  Returns false if the driver refuses.
inline bool encode_row_gather_map(void* tm_out, const void* base, size_t row_bytes, size_t rows) {
  typedef CUresult (*EncodeFn)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*, const cuuint64_t*,
                               const cuuint32_t*, const cuuint32_t*, CUtensorMapInterleave, CUtensorMapSwizzle,
                               CUtensorMapL2promotion, CUtensorMapFloatOOBfill);
  static EncodeFn enc = nullptr;
  if (!enc) {
    cudaDriverEntryPointQueryResult q;
    if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", (void**)&enc, cudaEnableDefault, &q) != cudaSuccess) enc = nullptr;
    if (!enc) return false;
  }
  const cuuint64_t gd[2] = {(cuuint64_t)row_bytes, (cuuint64_t)rows}, gs[1] = {(cuuint64_t)row_bytes};
  const cuuint32_t box[2] = {128, 1}, es[2] = {1, 1};
  return enc(reinterpret_cast<CUtensorMap*>(tm_out), CU_TENSOR_MAP_DATA_TYPE_UINT8, 2, const_cast<void*>(base), gd, gs, box, es,
             CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_128B, CU_TENSOR_MAP_L2_PROMOTION_L2_128B,
             CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE) == CUDA_SUCCESS;
}


// Host: 2D tensor map over a row-major [rows, cols] bf16 array for plain tiled loads of box_rows x 64
// elements (128 bytes per row) with the 128-byte swizzle — the SWIZZLE_128B K-major operand layout
// (8-row atoms of 1024 B).  Rows or columns beyond the array come back as zeros.
inline bool encode_tile_map_bf16(void* tm_out, const void* base, size_t rows, size_t cols, unsigned box_rows) {
  typedef CUresult (*EncodeFn)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*, const cuuint64_t*,
                               const cuuint32_t*, const cuuint32_t*, CUtensorMapInterleave, CUtensorMapSwizzle,
                               CUtensorMapL2promotion, CUtensorMapFloatOOBfill);
  static EncodeFn enc = nullptr;
  if (!enc) {
    cudaDriverEntryPointQueryResult q;
    if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", (void**)&enc, cudaEnableDefault, &q) != cudaSuccess) enc = nullptr;
    if (!enc) return false;
  }
  const cuuint64_t gd[2] = {(cuuint64_t)cols, (cuuint64_t)rows}, gs[1] = {(cuuint64_t)cols * 2};
  const cuuint32_t box[2] = {64, box_rows}, es[2] = {1, 1};
  return enc(reinterpret_cast<CUtensorMap*>(tm_out), CU_TENSOR_MAP_DATA_TYPE_BFLOAT16, 2, const_cast<void*>(base), gd, gs, box, es,
             CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_128B, CU_TENSOR_MAP_L2_PROMOTION_L2_256B,
             CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE) == CUDA_SUCCESS;
}
// box (c0 = first column, c1 = first row) of a tiled tensor map -> shared memory
__device__ __forceinline__ void tma_tile_2d(uint32_t dst, const CUtensorMap* tm, uint32_t bar, int c0, int c1) {
  asm volatile("cp.async.bulk.tensor.2d.shared::cluster.global.tile.mbarrier::complete_tx::bytes [%0], [%1, {%3, %4}], [%2];"
               ::"r"(dst), "l"(tm), "r"(bar), "r"(c0), "r"(c1)
               : "memory");
}

}  // namespace caee_umma
