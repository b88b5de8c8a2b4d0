// expert_fp8_wide.cu — S7 grouped SwiGLU expert FFN for FP8-E4M3 weights with 128x128 block
// scales at PREFILL sizes (BASELINE.json config 4's 4096-token batch) on sm_100a.
//
// Why a second e4m3 kernel.  With hundreds of tokens per expert the step sits on the ridge between
// the tensor pipe and HBM (3.25 TFLOP against 11.3 GB for config 4: 287 flop/B).  The decode
// kernel (expert_fp8.cu) feeds the e4m3 codes to kind::f8f6f4 as they are and therefore has to
// apply the per-(128x128) weight scale OUTSIDE the MMA: a fresh TMEM accumulator per 128-k block,
// promoted by the epilogue warps.  That is free at decode, but at N = 128 tokens the promotion
// reads 128 KB of TMEM per block at 64 B/clk — twice the time of the block's MMAs — and the
// two-term activations double the MMA work on top: 0.39 PFLOP/s.  Here the scale is folded into
// the weights instead: converter warps widen the e4m3 codes to fp16 (code x block scale x 2^J, one
// rounding to fp16's 11 bits; 2^J is the expert's power of two that puts its largest scale in
// [64, 128), so |code| <= 448 cannot overflow, see k_scale_norm in expert_fp8.cu), the MMAs are
// kind::f16 and accumulate over the WHOLE k range in TMEM; the epilogue runs once per tile and
// multiplies by 2^-J.  The token operand is fp16 too (tcgen05.mma kind::f16 with A = fp16 and
// B = bf16 is an illegal instruction): x is converted once per step by k_gather_x (exact for
// 6.1e-5 <= |x| <= 65504, clamped above), h is rounded to fp16 by the phase-1 epilogue.
//
// Tile shape.  Per CTA: 256 weight rows ([gate | up] of 128 features, or 256 down rows) x up to
// 256 tokens (one run; N = 256 is the widest tcgen05.mma), i.e. two 128 x 256 fp32 accumulators =
// all 512 TMEM columns, single-buffered.
//
// Token operand.  tile::gather4 row gathers (the decode kernels' way) cost ~20 cycles per
// 128-byte row in the TMA unit: at 256 rows per stage they, not the tensor pipe, paced the first
// version of this kernel.  So both token operands are kept as per-run STAGE IMAGES: for run r
// (rows padded to 16) stage s = the 64 k of every row, 128 bytes each, in 128-byte-swizzled
// 8-row atoms — ONE contiguous bulk copy per stage.  x's images are written once per step by
// k_gather_x (0.15 ms at 4096 tokens, bound by HBM writes: 0.5 GB at 3.2 TB/s, where a memset reaches 3.8); h's images are written in place by
// the phase-1 epilogue.  (Round 2 tried to drop k_gather_x by gathering the x rows inside this kernel with
// 16-byte cp.async copies from an fp16 copy of x — two loader warps, 2048 copies per stage, swizzled on the
// way in, cp.async.mbarrier.arrive on the stage barrier: correct, but the expert kernel went from 4.15 to
// 5.8 ms at 4096 tokens, so the images stay.)
//
// What bounds it.  Shared-memory bandwidth (128 B/clk): per 64 k the two MMAs read 32 KB of
// weights and 2 x 32 KB of tokens, the bulk copy writes 32 KB of tokens and the converters write
// 32 KB of fp16 — 160 KB for 1024 MMA cycles.  That is why the codes go global -> registers ->
// shared memory (no raw staging ring: it cost another 32 KB per 64 k).  The CTA-pair variant
// (template kPair, cta_group::2: each CTA of a pair reads half of the token operand, 112 KB per
// 64 k) is built and parity-tested but opt-in (CAEE_FP8_WIDE_PAIRS=1): on this pool's B200s both
// variants run into the 1000 W power cap (SM clock 1.6-1.9 GHz under load) and measure the same
// 4.0-4.2 ms for config 4's 4096-token step.
//
// Pipeline (640 threads, 1 CTA per SM; all rings are mbarrier full/empty pairs):
//   warp 0        tile claimer (atomic ticket, shared-memory queue; see umma_common.cuh)
//   warps 8-15    converters: packed e4m3 image (expert_fp8.cu's layout) -> registers -> 64-k fp16
//                 stages in the UMMA canonical K-major no-swizzle order (cvt ring, 3 x 32 KB)
//   warp 2        token-operand loader: one bulk copy per 64-k stage (tok ring, 4 x 32 KB)
//   warp 1        MMA issuer: 8 tcgen05.mma (M 128, N = padded tokens, K 16) per 64-k stage
//   warps 4-7, 16-19   epilogue: TMEM -> SwiGLU -> h (fp16), or -> o rows (fp32)
#include <cstdio>
#include <cstdlib>
#include <cstring>

#include "umma_common.cuh"

namespace {

using namespace caee_umma;

constexpr int kThreads = 640;
constexpr int kKRaw = 128;                 // k per raw stage = one block-scale block
constexpr int kKSub = 64;                  // k per converted / token stage
constexpr int kCvtStages = 3, kTokStages = 4;
constexpr int kCvtBytes = 2 * kTileRows * kKSub * 2;            // 32 KB: two 128-row bf16 tiles
constexpr int kTokBytes = CAEE_RUN_TOKENS_WIDE * kKSub * 2;     // 32 KB: 256 rows of 128 bytes
constexpr int kConvWarps = 8, kEpiWarps = 8, kLoadWarps = 1;
constexpr int kCvtOff = 0, kTokOff = kCvtOff + kCvtStages * kCvtBytes;
constexpr int kSmemBytes = kTokOff + kTokStages * kTokBytes;    // 224 KB
constexpr int kAccCols = 256;              // TMEM columns per accumulator
constexpr int kMaxKb = 64;                 // most 128-k blocks per tile: H, I <= 8192 (caee_fp8_wide_supported)
// The token operand is fp16 as well (x converted by k_gather_x, h written as fp16): kind::f16 takes
// fp16 or bf16 but not one of each (tcgen05.mma with A = fp16, B = bf16 is an illegal instruction).
constexpr bool kTokF16 = true;

struct WideParams {
  caee_worklist wl;
  uint8_t* const* packed;   // [E+S] e4m3 stage images + scale table (expert_fp8.cu's layout)
  const uint8_t* xg;        // token-operand stage images of x (k_gather_x), see "Token operand" above
  uint8_t* hbuf;            // the same for h, written by the phase-1 epilogue
  float* obuf;              // [T*(k+S),H]
  int H, I;
  int P1, P2, KB1, KB2;     // tiles per run and 128-k stages per tile, per phase
  int run_begin, run_count, ticket;
  int sc_off;               // byte offset of the scale table in a packed image
  int t2_off;               // float offset of its phase-2 part
  int norm_off;             // byte offset of the expert's {2^J, 2^-J} pair (expert_fp8.cu: k_scale_norm)
  int slots;                // k + S: an o row d belongs to token d / slots
};

// 16 e4m3 codes (one core-matrix row of the image) x scale -> 16 fp16, as two 8-element rows.
// s2 = the block scale x 2^J of the expert, twice: |code| <= 448 and s 2^J < 128 keep the products
// finite; a code's 4 significant bits x the scale's 11 round once, to fp16's 11.
__device__ __forceinline__ void widen16(const uint4 v, const __half2 s2, uint4& lo8, uint4& hi8) {
  const uint32_t w[4] = {v.x, v.y, v.z, v.w};
  uint32_t o[8];
#pragma unroll
  for (int i = 0; i < 4; ++i) {
    uint32_t h0, h1;
    asm("cvt.rn.f16x2.e4m3x2 %0, %1;" : "=r"(h0) : "h"((uint16_t)(w[i] & 0xffffu)));
    asm("cvt.rn.f16x2.e4m3x2 %0, %1;" : "=r"(h1) : "h"((uint16_t)(w[i] >> 16)));
    const __half2 p0 = __hmul2(*reinterpret_cast<const __half2*>(&h0), s2);
    const __half2 p1 = __hmul2(*reinterpret_cast<const __half2*>(&h1), s2);
    o[2 * i] = *reinterpret_cast<const uint32_t*>(&p0);
    o[2 * i + 1] = *reinterpret_cast<const uint32_t*>(&p1);
  }
  lo8 = make_uint4(o[0], o[1], o[2], o[3]);
  hi8 = make_uint4(o[4], o[5], o[6], o[7]);
}

// streaming 16-byte load of packed codes (read once per run: no L1 allocation)
__device__ __forceinline__ uint4 ldg_stream(const uint8_t* p) {
  uint4 v;
  asm volatile("ld.global.nc.L1::no_allocate.v4.b32 {%0,%1,%2,%3}, [%4];" : "=r"(v.x), "=r"(v.y), "=r"(v.z), "=r"(v.w) : "l"(p));
  return v;
}
__device__ __forceinline__ void sts128(uint32_t a, const uint4 v) {
  asm volatile("st.shared.v4.b32 [%0], {%1,%2,%3,%4};" ::"r"(a), "r"(v.x), "r"(v.y), "r"(v.z), "r"(v.w) : "memory");
}

#ifdef CAEE_WIDE_STATS
#define WAIT_T(acc, ...) do { long long _t0 = clock64(); __VA_ARGS__; acc += clock64() - _t0; } while (0)
#else
#define WAIT_T(acc, ...) do { __VA_ARGS__; } while (0)
#endif

// kPair: two CTAs of a cluster work on the same run with cta_group::2 MMAs (M = 256: each CTA
// brings the 128 + 128 weight rows of ITS feature block and HALF of the run's token rows), so a CTA
// reads 64 KB instead of 96 KB of operands per 64 k and fetches half of the token stage.  Tiles are
// then handed out statically (pair c takes pair-tiles c, c + pairs, ...: still phase-1 tiles first,
// in increasing order, so the phase-2 wait on a run's h cannot deadlock); the leader CTA (cluster
// rank 0) issues the MMAs and frees / fills the barriers of both CTAs with multicast commits, the
// peer's warp 1 forwards its "stage full" events to the leader.
template <bool kPair>
__global__ void __launch_bounds__(kThreads, 1) k_expert_fp8_wide(const __grid_constant__ WideParams p) {
  extern __shared__ __align__(1024) uint8_t smem_raw[];
  uint8_t* smem = reinterpret_cast<uint8_t*>((reinterpret_cast<uintptr_t>(smem_raw) + 1023) & ~(uintptr_t)1023);
  constexpr int kBars = 2 * (kCvtStages + kTokStages) + 2 + 2 * kQueue + kCvtStages + kTokStages;
  __shared__ __align__(8) uint64_t bars[kBars];
  __shared__ uint32_t tmem_base_s;
  __shared__ int tq_slots[kQueue];

  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const uint32_t smem_base = smem_u32(smem);
  const uint32_t cfull0 = smem_u32(&bars[0]), cempty0 = cfull0 + 8 * kCvtStages;
  const uint32_t kfull0 = cempty0 + 8 * kCvtStages, kempty0 = kfull0 + 8 * kTokStages;
  const uint32_t tfull = kempty0 + 8 * kTokStages, tempty = tfull + 8;
  const uint32_t qfull0 = tempty + 8, qempty0 = qfull0 + 8 * kQueue;
  const uint32_t pcr0 = qempty0 + 8 * kQueue, pkr0 = pcr0 + 8 * kCvtStages;   // leader: the peer's stage is full
  const uint32_t rank = kPair ? cluster_ctarank() : 0u;
  const TileMap tm{p.run_count >= 0 ? p.run_count : p.wl.meta[1], p.run_begin, kPair ? p.P1 / 2 : p.P1, kPair ? p.P2 / 2 : p.P2};
  int ti = (int)(blockIdx.x >> 1);                 // kPair: this pair's next pair-tile
  const int tstride = (int)(gridDim.x >> 1);
  (void)ti; (void)tstride;
// next tile of a role: popped from the ticket queue, or (pairs) the static schedule; sub = this CTA's feature block
#define NEXT_TILE(POP) (kPair ? (tm.at(ti, t) ? (ti += tstride, t.sub = 2 * t.sub + (int)rank, true) : false) : tm.at(POP, t))

  if (threadIdx.x == 0) {
    for (int s = 0; s < kCvtStages; ++s) {
      mbar_init(cfull0 + 8 * s, kConvWarps);
      mbar_init(cempty0 + 8 * s, 1);           // tcgen05.commit
    }
    for (int s = 0; s < kTokStages; ++s) {
      mbar_init(kfull0 + 8 * s, 1);            // expect_tx arrive of the loader
      mbar_init(kempty0 + 8 * s, 1);           // tcgen05.commit
    }
    mbar_init(tfull, 1);                       // tcgen05.commit
    mbar_init(tempty, kPair ? 2 * kEpiWarps : kEpiWarps);   // pairs: the leader waits for both CTAs' epilogues
    for (int s = 0; s < kCvtStages; ++s) mbar_init(pcr0 + 8 * s, 1);
    for (int s = 0; s < kTokStages; ++s) mbar_init(pkr0 + 8 * s, 1);
    for (int q = 0; q < kQueue; ++q) {
      mbar_init(qfull0 + 8 * q, 1);
      mbar_init(qempty0 + 8 * q, 1 + kLoadWarps + kEpiWarps + kConvWarps);
    }
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
  }
  if (warp == 2) {
    if (kPair) {
      asm volatile("tcgen05.alloc.cta_group::2.sync.aligned.shared::cta.b32 [%0], %1;" ::"r"(smem_u32(&tmem_base_s)), "n"(kTmemCols));
      asm volatile("tcgen05.relinquish_alloc_permit.cta_group::2.sync.aligned;");
    } else {
      asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], %1;" ::"r"(smem_u32(&tmem_base_s)), "n"(kTmemCols));
      asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;");
    }
  }
  tc_fence_before();
  __syncthreads();
  if (kPair) cluster_sync_all();               // both CTAs' barriers exist before any remote arrive / multicast commit
  tc_fence_after();
  const uint32_t tmem_base = tmem_base_s;
  TileQueue tq{qfull0, qempty0, tq_slots, 0, 0};
  Tile t;
  long long w_a = 0, w_b = 0, w_c = 0, w_d = 0, w_e = 0;   // wait cycles (CAEE_WIDE_STATS builds print them)
  const long long t_start = clock64();
  (void)t_start; (void)w_a; (void)w_b; (void)w_c; (void)w_d; (void)w_e;

  if (warp == 0) {
    // ===== tile claimer: one atomic ticket per tile, broadcast through the shared-memory queue
    if (!kPair && lane == 0) {
      int q = 0, qph = 0;
      for (;;) {
        WAIT_T(w_a, mbar_wait(qempty0 + 8 * q, qph ^ 1));
        const int i = atomicAdd(p.wl.sched + p.ticket, 1);
        tq_slots[q] = i;
        mbar_arrive(qfull0 + 8 * q);
        if (++q == kQueue) { q = 0; qph ^= 1; }
        if (!tm.at(i, t)) break;
      }
    }
  } else if (warp == 1 && rank == 0) {
    // ===== MMA issuer: fp16 x fp16, the accumulator pair lives in TMEM for the whole k range.
    // The whole warp runs the loop (uniform control flow); one elected lane issues.
    int cs = 0, cph = 0, ks = 0, kph = 0;
    const uint32_t d0 = tmem_base, d1 = tmem_base + kAccCols;
    for (int it = 0; NEXT_TILE(tq.pop()); ++it) {
      const int npad = (__shfl_sync(0xffffffffu, p.wl.run_n[t.run], 0) + 15) & ~15;
      // kind::f16, A and B fp16 (format 0), D fp32, both K-major; M = 128, or 256 over the CTA pair
      const uint32_t idesc = (1u << 4) | ((uint32_t)(npad >> 3) << 17) | ((uint32_t)((kPair ? 2 * kTileRows : kTileRows) >> 4) << 24);
      const int nsub = 2 * (t.phase == 1 ? p.KB1 : p.KB2);
      if (kPair) WAIT_T(w_a, mbar_wait_cluster(tempty, (it & 1) ^ 1));
      else WAIT_T(w_a, mbar_wait(tempty, (it & 1) ^ 1));
      tc_fence_after();
      for (int s = 0; s < nsub; ++s) {
        WAIT_T(w_b, mbar_wait(cfull0 + 8 * cs, cph));
        WAIT_T(w_c, mbar_wait(kfull0 + 8 * ks, kph));
        if (kPair) {
          WAIT_T(w_d, mbar_wait_cluster(pcr0 + 8 * cs, cph));
          WAIT_T(w_e, mbar_wait_cluster(pkr0 + 8 * ks, kph));
        }
        tc_fence_after();
        const uint32_t a_addr = smem_base + kCvtOff + cs * kCvtBytes;
        const uint64_t a0 = make_desc(a_addr), a1 = make_desc(a_addr + kATileBytes);
        const uint64_t b = make_desc_sw128(smem_base + kTokOff + ks * kTokBytes);
        if (elect_one()) {
          if (kPair) {
            if (s == 0) {
              umma_f16_pair_imm<false>(d0, a0, b, idesc);
              umma_f16_pair_imm<false>(d1, a1, b, idesc);
            } else {
              umma_f16_pair_imm<true>(d0, a0, b, idesc);
              umma_f16_pair_imm<true>(d1, a1, b, idesc);
            }
#pragma unroll
            for (int k16 = 1; k16 < kKSub / 16; ++k16) {
              umma_f16_pair_imm<true>(d0, a0 + (uint64_t)(k16 * 16), b + (uint64_t)(k16 * 2), idesc);
              umma_f16_pair_imm<true>(d1, a1 + (uint64_t)(k16 * 16), b + (uint64_t)(k16 * 2), idesc);
            }
            tc_commit_pair(cempty0 + 8 * cs);
            tc_commit_pair(kempty0 + 8 * ks);
            if (s == nsub - 1) tc_commit_pair(tfull);
          } else {
            if (s == 0) {
              umma_bf16_imm<false>(d0, a0, b, idesc);
              umma_bf16_imm<false>(d1, a1, b, idesc);
            } else {
              umma_bf16_imm<true>(d0, a0, b, idesc);
              umma_bf16_imm<true>(d1, a1, b, idesc);
            }
#pragma unroll
            for (int k16 = 1; k16 < kKSub / 16; ++k16) {   // per 16-element k-step: weights +256 B, tokens +32 B (>> 4)
              umma_bf16_imm<true>(d0, a0 + (uint64_t)(k16 * 16), b + (uint64_t)(k16 * 2), idesc);
              umma_bf16_imm<true>(d1, a1 + (uint64_t)(k16 * 16), b + (uint64_t)(k16 * 2), idesc);
            }
            tc_commit(cempty0 + 8 * cs);
            tc_commit(kempty0 + 8 * ks);
            if (s == nsub - 1) tc_commit(tfull);
          }
        }
        __syncwarp();
        if (++cs == kCvtStages) { cs = 0; cph ^= 1; }
        if (++ks == kTokStages) { ks = 0; kph ^= 1; }
      }
    }
  } else if (warp == 1 || (kPair && warp == 3 && rank != 0)) {
    // ===== (pairs, peer CTA) forwarders: this CTA's converted-weight stages (warp 1) and token
    // stages (warp 3) are full -> tell the leader, whose MMAs read them
    if (lane == 0) {
      const bool wts = warp == 1;
      const int depth = wts ? kCvtStages : kTokStages;
      const uint32_t src0 = wts ? cfull0 : kfull0, dst0 = wts ? pcr0 : pkr0;
      int st = 0, ph = 0;
      while (NEXT_TILE(0)) {
        const int nsub = 2 * (t.phase == 1 ? p.KB1 : p.KB2);
        for (int s = 0; s < nsub; ++s) {
          WAIT_T(w_b, mbar_wait(src0 + 8 * st, ph));
          mbar_arrive_remote(dst0 + 8 * st, 0);
          if (++st == depth) { st = 0; ph ^= 1; }
        }
      }
    }
  } else if (warp == 2) {
    // ===== token-operand loader: ONE bulk copy per 64-k stage from the run's stage images (x:
    // written by k_gather_x; h: written by the phase-1 epilogues), npad rows of 128 bytes
    if (lane == 0) {
      int stage = 0, ph = 0;
      while (NEXT_TILE(tq.pop1())) {
        const int npad = (p.wl.run_n[t.run] + 15) & ~15;
        const int nsub = 2 * (t.phase == 1 ? p.KB1 : p.KB2);
        const size_t row_bytes = (size_t)(t.phase == 1 ? p.H : p.I) * 2;
        const uint32_t stage_bytes = (uint32_t)npad * 128u;
        const uint32_t bytes = kPair ? stage_bytes / 2 : stage_bytes;      // pairs: this CTA's half of the rows
        const uint8_t* src = (t.phase == 1 ? p.xg : p.hbuf) + (size_t)p.wl.run_hrow[t.run] * row_bytes + (kPair ? rank * bytes : 0u);
        if (t.phase == 2) {
          // h of this run is complete once all P1 gate/up tiles have published it (generic-proxy
          // stores of other SMs, read here through the async proxy)
          const int* flag = p.wl.ready + t.run;
          WAIT_T(w_b, while (ld_acquire(flag) < p.P1) __nanosleep(64));
          asm volatile("fence.proxy.async;" ::: "memory");
        }
        for (int s = 0; s < nsub; ++s) {
          WAIT_T(w_a, mbar_wait(kempty0 + 8 * stage, ph ^ 1));
          mbar_arrive_expect_tx(kfull0 + 8 * stage, bytes);
          bulk_g2s(smem_base + kTokOff + stage * kTokBytes, src + (size_t)s * stage_bytes, bytes, kfull0 + 8 * stage);
          if (++stage == kTokStages) { stage = 0; ph ^= 1; }
        }
      }
    }
  } else if (warp == 3) {
    // spare warp
  } else if (warp < 8 || warp >= 16) {
    // ===== epilogue (warps 4-7 and 16-19): TMEM -> registers -> SwiGLU -> h (phase 1) or -> o rows
    // (phase 2).  Two warps per TMEM lane quadrant q = warp % 4, each one half of the token columns.
    const int q = warp & 3, eh = warp >= 16;
    for (int it = 0; NEXT_TILE(tq.pop()); ++it) {
      const int n = p.wl.run_n[t.run], start = p.wl.run_start[t.run];
      const int npad = (n + 15) & ~15;
      const int half = (((npad >> 4) + 1) >> 1) << 4;
      const int c_lo = eh ? half : 0, c_hi = eh ? n : min(half, n);
      // phase 2: the o row of this warp's token columns, fetched before the accumulator is ready
      // (lane l holds columns c_lo + l, c_lo + l + 32, ...; broadcast by shuffle below)
      int dst_l[CAEE_RUN_TOKENS_WIDE / 64];
      if (t.phase == 2) {
#pragma unroll
        for (int i = 0; i < CAEE_RUN_TOKENS_WIDE / 64; ++i) {
          const int col = c_lo + i * 32 + lane;
          dst_l[i] = col < c_hi ? p.wl.ent_dst[start + col] : 0;
        }
      }
      const float inv = __ldg(reinterpret_cast<const float*>(p.packed[p.wl.run_expert[t.run]] + p.norm_off) + 1);   // 2^-J
      WAIT_T(w_a, mbar_wait(tfull, it & 1));
      tc_fence_after();
      const uint32_t tbase = tmem_base + ((uint32_t)(q * 32) << 16);
      const int row = q * 32 + lane;
      if (t.phase == 1) {
        // h[token c, feature f], f = 128 sub + row, goes to stage f / 64 of the run's h image:
        // row c of 128 bytes, 16-byte chunk (f % 64) / 8 at position chunk ^ (c % 8) (128-byte swizzle)
        const int f = t.sub * kTileRows + row;
        uint8_t* hrun = p.hbuf + (size_t)p.wl.run_hrow[t.run] * p.I * 2 + (size_t)(f >> 6) * npad * 128 + (f & 7) * 2;
        const int chunk = (f & 63) >> 3;
        for (int c = c_lo; c < c_hi; c += 16) {
          uint32_t g[16], u[16];
          tmem_ld16(tbase + c, g);
          tmem_ld16(tbase + kAccCols + c, u);
          tmem_ld_wait();
#pragma unroll
          for (int j = 0; j < 16; ++j) {
            if (c + j < c_hi) {
              const float gv = __uint_as_float(g[j]) * inv, uv = __uint_as_float(u[j]) * inv;
              // fp16 token operand: clamp like x (|h| > 65504 would become inf and then NaN in y)
              const float hv = fminf(fmaxf(__fdividef(gv, 1.0f + __expf(-gv)) * uv, -65504.f), 65504.f);
              const int cc = c + j;
              *reinterpret_cast<uint16_t*>(hrun + cc * 128 + ((chunk ^ (cc & 7)) << 4)) =
                  kTokF16 ? __half_as_ushort(__float2half_rn(hv)) : __bfloat16_as_ushort(__float2bfloat16_rn(hv));
            }
          }
        }
      } else {
        float* ocol = p.obuf + t.sub * 2 * kTileRows + row;
        for (int c = c_lo; c < c_hi; c += 16) {
          uint32_t v0[16], v1[16];
          tmem_ld16(tbase + c, v0);
          tmem_ld16(tbase + kAccCols + c, v1);
          tmem_ld_wait();
          const int rel = c - c_lo;
          int dsel = 0;
#pragma unroll
          for (int i = 0; i < CAEE_RUN_TOKENS_WIDE / 64; ++i)
            if ((rel >> 5) == i) dsel = dst_l[i];
#pragma unroll
          for (int j = 0; j < 16; ++j) {
            const int d = __shfl_sync(0xffffffffu, dsel, (rel & 31) + j);
            if (c + j < c_hi) {
              float* o = caee_o_base(p.wl, p.obuf, d / p.slots) + (ocol - p.obuf) + (size_t)d * p.H;
              o[0] = __uint_as_float(v0[j]) * inv;
              o[kTileRows] = __uint_as_float(v1[j]) * inv;
            }
          }
        }
      }
      tc_fence_before();
      __syncwarp();
      if (lane == 0) {
        if (kPair && rank != 0) mbar_arrive_remote(tempty, 0);
        else mbar_arrive(tempty);
      }
      if (t.phase == 1) {
        // publish this tile's slice of h: all 256 epilogue threads' stores (read later through the
        // async proxy by other SMs' bulk copies), then one release add
        asm volatile("fence.proxy.async;" ::: "memory");
        __threadfence();
        asm volatile("bar.sync 1, 256;" ::: "memory");
        if (threadIdx.x == 128) atomicAdd(p.wl.ready + t.run, 1);
      }
    }
  } else {
    // ===== converters (warps 8-15): e4m3 codes x block scale -> fp16, one 128-k stage -> two 64-k stages.
    // A 64-k half of a raw stage is 1024 chunks of 16 codes (2 tiles x 16 row groups x 4 k chunks x
    // 8 rows); chunk id = i * 256 + ct with i = 0..3, so i >> 1 is the tile half (its own scale),
    // a warp reads 512 contiguous bytes and writes 4 x 128 contiguous bytes twice.
    const int ct = threadIdx.x - 256;
    const int r8 = ct & 7, c4 = (ct >> 3) & 3;
    // byte offset of this thread's chunk i of half hh inside a 32 KB stage of the packed image
    // (= the offset of its first fp16 row inside a converted stage, with c4 doubled)
    int off_i[4];
#pragma unroll
    for (int i = 0; i < 4; ++i) off_i[i] = (i >> 1) * kATileBytes + (((i & 1) * 256 + ct) >> 5) * 1024 + r8 * 16;
    int cs = 0, cph = 0;
    while (NEXT_TILE(tq.pop())) {
      const int nkb = t.phase == 1 ? p.KB1 : p.KB2;
      const uint8_t* img = p.packed[p.wl.run_expert[t.run]];
      const float* tab = reinterpret_cast<const float*>(img + p.sc_off);
      const float* wsc = t.phase == 1 ? tab + (size_t)t.sub * p.KB1 * 2 : tab + p.t2_off + (size_t)t.sub * p.KB2 * 2;
      const uint8_t* src = img + (t.phase == 1 ? (size_t)t.sub * p.KB1 : (size_t)p.P1 * p.KB1 + (size_t)t.sub * p.KB2) * kAStageBytes + c4 * 128;
      const float nrm = __ldg(reinterpret_cast<const float*>(img + p.norm_off));
      // the tile's block scales, fetched once: lane l keeps those of k blocks l, l + 32, ... (a load per
      // k block in the loop below ends up next to its use and exposes its latency every 128 k)
      float sc0[kMaxKb / 32], sc1[kMaxKb / 32];
#pragma unroll
      for (int j = 0; j < kMaxKb / 32; ++j) {
        const int kbj = lane + 32 * j;
        sc0[j] = kbj < nkb ? __ldg(wsc + 2 * kbj) * nrm : 0.f;
        sc1[j] = kbj < nkb ? __ldg(wsc + 2 * kbj + 1) * nrm : 0.f;
      }
      // the codes go global -> registers (no shared-memory staging: shared-memory bandwidth is the
      // bound of this kernel): both 64-k halves of stage kb + 1 are in flight while stage kb is widened
      uint4 va[4], vb[4];
#pragma unroll
      for (int i = 0; i < 4; ++i) {
        va[i] = ldg_stream(src + off_i[i]);
        vb[i] = ldg_stream(src + off_i[i] + 512);
      }
      for (int kb = 0; kb < nkb; ++kb) {
        float s0 = 0.f, s1 = 0.f;
#pragma unroll
        for (int j = 0; j < kMaxKb / 32; ++j)
          if ((kb >> 5) == j) { s0 = sc0[j]; s1 = sc1[j]; }
        const __half2 w0 = __float2half2_rn(__shfl_sync(0xffffffffu, s0, kb & 31));
        const __half2 w1 = __float2half2_rn(__shfl_sync(0xffffffffu, s1, kb & 31));
        const uint8_t* nxt = src + (size_t)(kb + 1) * kAStageBytes;
#pragma unroll
        for (int hh = 0; hh < 2; ++hh) {
          // the commit that completed this barrier ordered the MMAs' reads of the stage before it; no
          // tcgen05.fence here: it would also wait for the code loads in flight for the next stage
          WAIT_T(w_b, mbar_wait(cempty0 + 8 * cs, cph ^ 1));
          const uint32_t dst = smem_base + kCvtOff + cs * kCvtBytes + c4 * 256;
#pragma unroll
          for (int i = 0; i < 4; ++i) {
            uint4 lo8, hi8;
            widen16(hh ? vb[i] : va[i], (i >> 1) ? w1 : w0, lo8, hi8);
            sts128(dst + off_i[i], lo8);
            sts128(dst + off_i[i] + 128, hi8);
          }
          if (kb + 1 < nkb) {
#pragma unroll
            for (int i = 0; i < 4; ++i) {
              if (hh) vb[i] = ldg_stream(nxt + off_i[i] + 512);
              else va[i] = ldg_stream(nxt + off_i[i]);
            }
          }
          fence_proxy_async_smem();
          __syncwarp();
          if (lane == 0) mbar_arrive(cfull0 + 8 * cs);
          if (++cs == kCvtStages) { cs = 0; cph ^= 1; }
        }
      }
    }
  }

#ifdef CAEE_WIDE_STATS
  if (lane == 0 && (blockIdx.x == 0 || blockIdx.x == 101) && (warp <= 3 || warp == 4 || warp == 8 || warp == 16))
    printf("cta %d warp %d: total %lld  wait a %lld b %lld c %lld d %lld e %lld\n", blockIdx.x, warp, clock64() - t_start, w_a, w_b, w_c, w_d, w_e);
#endif
#undef NEXT_TILE
  tc_fence_before();
  __syncthreads();
  if (kPair) cluster_sync_all();               // the peer's shared memory and TMEM stay until the leader's MMAs are done
  if (warp == 2) {
    tc_fence_after();
    if (kPair) asm volatile("tcgen05.dealloc.cta_group::2.sync.aligned.b32 %0, %1;" ::"r"(tmem_base), "n"(kTmemCols));
    else asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;" ::"r"(tmem_base), "n"(kTmemCols));
  }
}

// bf16 pair -> fp16 pair, clamped to fp16's range
__device__ __forceinline__ uint4 bf16x8_to_f16x8(uint4 v) {
  uint32_t* w = reinterpret_cast<uint32_t*>(&v);
#pragma unroll
  for (int q = 0; q < 4; ++q) {
    const float lo = __uint_as_float(w[q] << 16), hi = __uint_as_float(w[q] & 0xffff0000u);
    const __half2 h2 = __floats2half2_rn(fminf(fmaxf(lo, -65504.f), 65504.f), fminf(fmaxf(hi, -65504.f), 65504.f));
    w[q] = *reinterpret_cast<const uint32_t*>(&h2);
  }
  return v;
}

// x rows of every run -> the run's token-operand stage images (fp16).  CTA (r, y): run r, the y-th
// share of its 64-k stages, ALL rows: eight threads share a row's 128-byte piece (one 16-byte chunk
// each), the CTA covers 32 rows per pass, so a stage image (npad x 128 bytes) and the stages after it
// are written front to back — one contiguous region per CTA; rows >= n are written as zeros.
constexpr int kGatherY = 8, kGatherPass = CAEE_RUN_TOKENS_WIDE / 32;
__global__ void __launch_bounds__(256) k_gather_x(caee_worklist wl, const uint4* __restrict__ x, uint8_t* __restrict__ xg, int H,
                                                  int n_runs_arg) {
  const int n_runs = n_runs_arg >= 0 ? n_runs_arg : wl.meta[1];
  const int run = blockIdx.x;
  if (run >= n_runs) return;
  const int n = wl.run_n[run], start = wl.run_start[run], npad = (n + 15) & ~15;
  const int nsub = H / kKSub, j = threadIdx.x & 7, r0 = threadIdx.x >> 3;
  const int per = (nsub + gridDim.y - 1) / gridDim.y, s_lo = blockIdx.y * per, s_hi = min(nsub, s_lo + per);
  uint8_t* img = xg + (size_t)wl.run_hrow[run] * H * 2;
  const size_t sstride = (size_t)npad * 128;
  const uint4* src[kGatherPass];
  uint32_t doff[kGatherPass];
#pragma unroll
  for (int q = 0; q < kGatherPass; ++q) {
    const int rr = q * 32 + r0;
    src[q] = rr < n ? x + (size_t)wl.ent_tok[start + rr] * (H / 8) + j : nullptr;
    doff[q] = (uint32_t)((rr >> 3) * 1024 + (rr & 7) * 128 + ((j ^ (rr & 7)) << 4));
  }
  const int npass = (npad + 31) >> 5;
  for (int s = s_lo; s < s_hi; ++s) {
    uint4 v[kGatherPass];
#pragma unroll
    for (int q = 0; q < kGatherPass; ++q) {
      v[q] = make_uint4(0, 0, 0, 0);
      if (q < npass && src[q]) v[q] = __ldg(src[q] + s * 8);
    }
#pragma unroll
    for (int q = 0; q < kGatherPass; ++q)
      if (q < npass && q * 32 + r0 < npad) *reinterpret_cast<uint4*>(img + s * sstride + doff[q]) = bf16x8_to_f16x8(v[q]);
  }
}

}  // namespace

bool caee_fp8_wide_supported(const caee_ctx* c) { return c->d.H <= kMaxKb * kKRaw && c->d.I <= kMaxKb * kKRaw; }

size_t caee_fp8_wide_xg_bytes(const caee_ctx* c) { return c->h_rows_cap * (size_t)c->d.H * 2; }

// Once per step, after the work list is built: the x rows of every run, laid out for bulk copies.
void caee_launch_fp8_wide_prepare(caee_ctx* c, const void* x, int T, cudaStream_t st) {
  if (T <= 0) return;
  ++c->n_launches;
  k_gather_x<<<dim3((unsigned)c->wl.max_runs, kGatherY), 256, 0, st>>>(c->wl, (const uint4*)x, c->xg, c->d.H, -1);
}

// runs [run_begin, run_begin + run_count) (run_count < 0: every run of the work list), tile
// tickets from wl.sched[ticket].  Runs hold up to CAEE_RUN_TOKENS_WIDE tokens.
void caee_launch_expert_fp8_wide(caee_ctx* c, int T, int run_begin, int run_count, int ticket, cudaStream_t st) {
  (void)T;
  ++c->n_launches;
  const caee_layer_desc& d = c->d;
  WideParams p;
  p.wl = c->wl;
  p.packed = c->packed.dev_ptrs;
  p.xg = c->xg;
  p.hbuf = (uint8_t*)c->hbuf_b16;
  p.obuf = c->obuf;
  p.H = d.H; p.I = d.I;
  p.P1 = d.I / kTileRows; p.P2 = d.H / (2 * kTileRows);
  p.KB1 = d.H / kKRaw; p.KB2 = d.I / kKRaw;
  p.run_begin = run_begin; p.run_count = run_count; p.ticket = ticket;
  p.sc_off = (int)((size_t)3 * d.H * d.I);
  p.t2_off = p.P1 * p.KB1 * 2;
  p.norm_off = (int)caee_fp8_norm_offset(c);
  p.slots = d.k + d.S;
  if (!(c->attr_done & 4u)) {
    cudaFuncSetAttribute(k_expert_fp8_wide<false>, cudaFuncAttributeMaxDynamicSharedMemorySize, kSmemBytes + 1024);
    cudaFuncSetAttribute(k_expert_fp8_wide<true>, cudaFuncAttributeMaxDynamicSharedMemorySize, kSmemBytes + 1024);
    c->attr_done |= 4u;
  }
  // CTA pairs (cta_group::2) need an even number of tiles per run in both phases
  // (opt-in, caee_ctx::fp8_wide_pairs: on this pool's B200s the kernel runs into the 1000 W power cap
  // either way and the pair variant measures the same 4.0-4.2 ms; the single-CTA variant keeps the
  // dynamic tile tickets)
  if (c->fp8_wide_pairs && p.P1 % 2 == 0 && p.P2 % 2 == 0 && c->num_sms >= 2) {
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = dim3((unsigned)(c->num_sms & ~1));
    cfg.blockDim = dim3(kThreads);
    cfg.dynamicSmemBytes = kSmemBytes + 1024;
    cfg.stream = st;
    cudaLaunchAttribute at[1];
    at[0].id = cudaLaunchAttributeClusterDimension;
    at[0].val.clusterDim.x = 2; at[0].val.clusterDim.y = 1; at[0].val.clusterDim.z = 1;
    cfg.attrs = at; cfg.numAttrs = 1;
    // the static schedule needs every pair resident at once (a phase-2 tile waits for phase-1 tiles of other pairs)
    int max_pairs = c->wide_max_pairs;
    if (max_pairs < 0 && cudaOccupancyMaxActiveClusters(&max_pairs, k_expert_fp8_wide<true>, &cfg) != cudaSuccess) { max_pairs = 0; cudaGetLastError(); }
    c->wide_max_pairs = max_pairs;
    if (max_pairs * 2 >= (int)cfg.gridDim.x) {
      cudaLaunchKernelEx(&cfg, k_expert_fp8_wide<true>, p);
      return;
    }
  }
  k_expert_fp8_wide<false><<<c->num_sms, kThreads, kSmemBytes + 1024, st>>>(p);
}
