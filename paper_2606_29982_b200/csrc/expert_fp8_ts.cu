// expert_fp8_ts.cu — S7 grouped SwiGLU expert FFN for FP8-E4M3 weights with 128x128 block scales at
// PREFILL sizes, with the widened weights fed to the tensor cores from TENSOR MEMORY ("TS" MMAs:
// tcgen05.mma with the A operand in TMEM).
//
// Why a third e4m3 kernel.  expert_fp8_wide.cu widens the e4m3 codes to fp16 (code x block scale, one
// rounding; see there for the arithmetic, which this kernel shares) into SHARED memory and is bound by
// shared-memory bandwidth: per 64 k the converters write 32 KB, the MMAs read those 32 KB back plus the
// token operand twice, the bulk copy writes the tokens — 160 KB against the 128 KB that 1024 MMA cycles
// allow at N = 256, and the 64 KB of weight traffic does not shrink with the run (112 KB against 512
// MMA cycles at N = 128: tensor pipe 42-48% busy, profiles/r02_prefill_c4_T4096.md).  tcgen05.mma takes
// its A operand from tensor memory as well, so here the converter warps put the widened weights
// straight into TMEM with tcgen05.st (row = TMEM lane, two fp16 per 32-bit column — the layout a
// K-major A fragment has there) and the MMAs read them on the tensor datapath: shared memory carries
// only the token operand (48 KB per 64 k at N = 128, 375 cycles against 512 of MMAs).
//
// TMEM budget (512 columns), two shapes (TsCfg below).  192-token runs, the default: two fp32 accumulators of
// N <= 192 columns (gate | up of 128 features, or 256 down rows) = 384 columns, and an A ring of 2 stages x (2 tiles
// x 32 columns = 64 k of 128 rows each) = 128 columns.  128-token runs (CAEE_TS_RUN_TOKENS=128; round 2's first
// version): accumulators 256 columns, A ring 2 stages x 128 k = 256 columns.  A hot expert's weights are streamed
// (from L2) and converted once per run — conversion is cheap (F2FP + HMUL2 per code pair at full ALU rate), it was
// its shared-memory traffic that cost in expert_fp8_wide.cu — but a run costs 2.4-3.4 us whatever its length, so the
// longer runs win: config 4's 4096-token step has 354 runs instead of 433 and the kernel takes 3.41-3.45 instead of
// 3.57-3.62 ms (0.67-0.68 instead of 0.64-0.65 of the sustained tensor rate; same box, interleaved).
//
// Pipeline (640 threads, 1 CTA per SM; all rings are mbarrier full/empty pairs):
//   warp 0        tile claimer (atomic ticket, shared-memory queue; see umma_common.cuh) and weight producer: one
//                 32 KB bulk copy per 128-k stage of the packed e4m3 image (raw ring, 3 x 32 KB).  The first
//                 version of this kernel loaded the codes global -> registers in the converter threads, one
//                 stage ahead: 32 KB in flight per SM against the ~32 B/clk x ~1000 clk the stream needs, and
//                 the MMA warp waited 25% of the time for converted weights; the copy engine prefetches deeper
//                 at no register cost, and shared memory has room here (80 KB of traffic per 64 k at N = 128)
//   warps 8-15    converters: warp w owns TMEM lane quadrant w % 4 of tile half (w - 8) / 4; thread = one
//                 weight row: 128 codes per 128-k raw stage shared -> registers -> fp16 -> 2 x tcgen05.st (one A stage each,
//                 or both into one 128-k A stage)
//   warp 2        token-operand loader: one bulk copy per token stage from the run's stage image (tok ring, 5 x 24 KB
//                 of 64 k, or 4 x 32 KB of 128 k in the 128-token shape; x images by k_gather_x, h images by the phase-1 epilogue: expert_fp8_wide.cu).
//                 (Tried: writing the x images inside this kernel with the idle warp 3 of every CTA, row b of every
//                 run by CTA b, phase-1 tiles waiting on a per-run counter — parity green, but one warp per SM moves a
//                 14 KB row in ~20 us and the step went from 3.55 to 8.45 ms; k_gather_x stays.)
//   warp 1        MMA issuer: 8 tcgen05.mma (A from TMEM, M 128, N = padded tokens, K 16) per 64-k stage (16 per 128-k stage)
//   warps 4-7, 16-19   epilogue: TMEM -> SwiGLU -> h (fp16 stage image), or -> o rows (fp32)
#include <cstdio>
#include <cstring>

#include "umma_common.cuh"

namespace {

using namespace caee_umma;

constexpr int kThreads = 640;
constexpr int kKRaw = 128;                 // k per packed stage = one block-scale block
constexpr int kRawStages = 3;
constexpr int kConvWarps = 8, kEpiWarps = 8;
constexpr int kMaxKb = 64;
// Two shapes of the same kernel, by the most tokens of a run (= the MMAs' N, = TMEM columns per accumulator):
//   kRun 128: accumulators 2 x 128 columns, A ring 2 stages x 128 columns (128 k: one hand-over per block-scale block),
//             token ring 4 x 32 KB (128-k stages);
//   kRun 192: accumulators 2 x 192 columns, A ring 2 stages x 64 columns (64 k), token ring 5 x 24 KB (64-k stages).
//             A hot expert's image is streamed from L2 and converted once per 192 instead of once per 128 tokens
//             (config 4's 4096-token step: 354 runs instead of 433; a run costs 2.4-3.4 us whatever its length).
template <int kRun>
struct TsCfg {
  static constexpr int kSubK = kRun <= 128 ? 128 : 64;            // k per A stage and per token stage
  static constexpr int kAStagesT = 2;
  static constexpr int kTokStages = kRun <= 128 ? 4 : 5;
  static constexpr int kTokBytes = kRun * kSubK * 2;              // kSubK / 64 images of kRun rows x 128 bytes
  static constexpr int kRawOff = kTokStages * kTokBytes;          // raw ring behind the token ring
  static constexpr int kSmemBytes = kRawOff + kRawStages * kAStageBytes;   // 224 KB / 216 KB
  static constexpr int kAccCols = kRun;                           // TMEM columns per accumulator
  static constexpr int kACol0 = 2 * kAccCols;                     // first column of the A ring
  static constexpr int kAStageCols = kSubK;                       // two tiles x kSubK / 2 columns (two fp16 per column)
  static_assert(kACol0 + kAStagesT * kAStageCols <= kTmemCols, "TMEM budget");
  static_assert(kSmemBytes + 1024 <= 227 * 1024, "shared memory budget");
};

struct TsParams {
  caee_worklist wl;
  uint8_t* const* packed;   // [E+S] e4m3 stage images + scale table (expert_fp8.cu's layout)
  const uint8_t* xg;        // token-operand stage images of x (k_gather_x)
  uint8_t* hbuf;            // the same for h, written by the phase-1 epilogue
  float* obuf;              // [T*(k+S),H]
  int H, I;
  int P1, P2, KB1, KB2;     // tiles per run and 128-k stages per tile, per phase
  int run_begin, run_count, ticket;
  int sc_off, t2_off, norm_off;   // as in expert_fp8_wide.cu
  int slots;                // k + S
};

// 16 e4m3 codes x scale -> 16 fp16 as 8 packed words, k ascending (expert_fp8_wide.cu: widen16)
__device__ __forceinline__ void widen16_ts(const uint4 v, const __half2 s2, uint32_t* o) {
  const uint32_t w[4] = {v.x, v.y, v.z, v.w};
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
}
// 32 consecutive 32-bit columns of this thread's TMEM lane
__device__ __forceinline__ void tmem_st32(uint32_t taddr, const uint32_t (&v)[32]) {
  asm volatile(
      "tcgen05.st.sync.aligned.32x32b.x32.b32 [%0], {%1,%2,%3,%4,%5,%6,%7,%8,%9,%10,%11,%12,%13,%14,%15,%16,%17,%18,%19,%20,%21,%22,%23,%24,%25,"
      "%26,%27,%28,%29,%30,%31,%32};" ::"r"(taddr),
      "r"(v[0]), "r"(v[1]), "r"(v[2]), "r"(v[3]), "r"(v[4]), "r"(v[5]), "r"(v[6]), "r"(v[7]), "r"(v[8]), "r"(v[9]), "r"(v[10]), "r"(v[11]),
      "r"(v[12]), "r"(v[13]), "r"(v[14]), "r"(v[15]), "r"(v[16]), "r"(v[17]), "r"(v[18]), "r"(v[19]), "r"(v[20]), "r"(v[21]), "r"(v[22]),
      "r"(v[23]), "r"(v[24]), "r"(v[25]), "r"(v[26]), "r"(v[27]), "r"(v[28]), "r"(v[29]), "r"(v[30]), "r"(v[31])
      : "memory");
}
__device__ __forceinline__ void tmem_st_wait() { asm volatile("tcgen05.wait::st.sync.aligned;" ::: "memory"); }
// D[tmem] (+)= A[tmem] * B[smem]^T, kind::f16, M = 128, K = 16
template <bool kAcc>
__device__ __forceinline__ void umma_f16_ts(uint32_t d_tmem, uint32_t a_tmem, uint64_t b_desc, uint32_t idesc) {
  asm volatile(
      "{\n\t.reg .pred p;\n\t"
      "setp.ne.b32 p, %4, 0;\n\t"
      "tcgen05.mma.cta_group::1.kind::f16 [%0], [%1], %2, %3, p;\n\t}" ::"r"(d_tmem),
      "r"(a_tmem), "l"(b_desc), "r"(idesc), "n"(kAcc ? 1 : 0)
      : "memory");
}

#ifdef CAEE_WIDE_STATS
#define WAIT_T(acc, ...) do { long long _t0 = clock64(); __VA_ARGS__; acc += clock64() - _t0; } while (0)
#else
#define WAIT_T(acc, ...) do { __VA_ARGS__; } while (0)      /* acc is not even named in the product build */
#endif

template <int kRun>
__global__ void __launch_bounds__(kThreads, 1) k_expert_fp8_ts(const __grid_constant__ TsParams p) {
  using C = TsCfg<kRun>;
  constexpr int kSubK = C::kSubK, kAStagesT = C::kAStagesT, kTokStages = C::kTokStages, kTokBytes = C::kTokBytes;
  constexpr int kRawOff = C::kRawOff, kAccCols = C::kAccCols, kACol0 = C::kACol0, kAStageCols = C::kAStageCols;
  constexpr int kRunTokens = kRun;
  extern __shared__ __align__(1024) uint8_t smem_raw[];
  uint8_t* smem = reinterpret_cast<uint8_t*>((reinterpret_cast<uintptr_t>(smem_raw) + 1023) & ~(uintptr_t)1023);
  constexpr int kBars = 2 * (kAStagesT + kTokStages + kRawStages) + 2 + 2 * kQueue;
  __shared__ __align__(8) uint64_t bars[kBars];
  __shared__ uint32_t tmem_base_s;
  __shared__ int tq_slots[kQueue];

  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const uint32_t smem_base = smem_u32(smem);
  const uint32_t cfull0 = smem_u32(&bars[0]), cempty0 = cfull0 + 8 * kAStagesT;
  const uint32_t kfull0 = cempty0 + 8 * kAStagesT, kempty0 = kfull0 + 8 * kTokStages;
  const uint32_t tfull = kempty0 + 8 * kTokStages, tempty = tfull + 8;
  const uint32_t qfull0 = tempty + 8, qempty0 = qfull0 + 8 * kQueue;
  const uint32_t rfull0 = qempty0 + 8 * kQueue, rempty0 = rfull0 + 8 * kRawStages;
  const TileMap tm{p.run_count >= 0 ? p.run_count : p.wl.meta[1], p.run_begin, p.P1, p.P2};

  if (threadIdx.x == 0) {
    for (int s = 0; s < kAStagesT; ++s) {
      mbar_init(cfull0 + 8 * s, kConvWarps);   // one lane of each converter warp
      mbar_init(cempty0 + 8 * s, 1);           // tcgen05.commit
    }
    for (int s = 0; s < kTokStages; ++s) {
      mbar_init(kfull0 + 8 * s, 1);            // expect_tx arrive of the loader
      mbar_init(kempty0 + 8 * s, 1);           // tcgen05.commit
    }
    for (int s = 0; s < kRawStages; ++s) {
      mbar_init(rfull0 + 8 * s, 1);            // expect_tx arrive of the producer
      mbar_init(rempty0 + 8 * s, kConvWarps);  // one lane of each converter warp
    }
    mbar_init(tfull, 1);                       // tcgen05.commit
    mbar_init(tempty, kEpiWarps);
    for (int q = 0; q < kQueue; ++q) {
      mbar_init(qfull0 + 8 * q, 1);
      mbar_init(qempty0 + 8 * q, 2 + kEpiWarps + kConvWarps);   // MMA warp + loader + epilogue + converter warps
    }
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
  }
  if (warp == 2) {
    asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], %1;" ::"r"(smem_u32(&tmem_base_s)), "n"(kTmemCols));
    asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;");
  }
  tc_fence_before();
  __syncthreads();
  tc_fence_after();
  const uint32_t tmem_base = tmem_base_s;
  TileQueue tq{qfull0, qempty0, tq_slots, 0, 0};
  Tile t;
#ifdef CAEE_WIDE_STATS
  long long w_a = 0, w_b = 0, w_c = 0, w_d = 0;   // wait cycles of this thread, printed at the end
  const long long t_start = clock64();
#endif

  if (warp == 0) {
    // ===== tile claimer and weight producer: one atomic ticket per tile, broadcast through the shared-memory queue;
    // one 32 KB bulk copy per 128-k stage of the tile's packed e4m3 codes
    if (lane == 0) {
      int q = 0, qph = 0, stage = 0, ph = 0;
      for (;;) {
        mbar_wait(qempty0 + 8 * q, qph ^ 1);
        const int i = atomicAdd(p.wl.sched + p.ticket, 1);
        tq_slots[q] = i;
        mbar_arrive(qfull0 + 8 * q);
        if (++q == kQueue) { q = 0; qph ^= 1; }
        if (!tm.at(i, t)) break;
        const int nkb = t.phase == 1 ? p.KB1 : p.KB2;
        const uint8_t* src = p.packed[p.wl.run_expert[t.run]] +
                             (t.phase == 1 ? (size_t)t.sub * p.KB1 : (size_t)p.P1 * p.KB1 + (size_t)t.sub * p.KB2) * kAStageBytes;
        for (int kb = 0; kb < nkb; ++kb) {
          mbar_wait(rempty0 + 8 * stage, ph ^ 1);
          mbar_arrive_expect_tx(rfull0 + 8 * stage, kAStageBytes);
          bulk_g2s(smem_base + kRawOff + stage * kAStageBytes, src + (size_t)kb * kAStageBytes, kAStageBytes, rfull0 + 8 * stage);
          if (++stage == kRawStages) { stage = 0; ph ^= 1; }
        }
      }
    }
  } else if (warp == 1) {
    // ===== MMA issuer: fp16 x fp16, A from the TMEM ring, the accumulator pair lives in TMEM for the whole
    // k range.  The whole warp runs the loop (uniform control flow); one elected lane issues.
    int cs = 0, cph = 0, ks = 0, kph = 0;
    const uint32_t d0 = tmem_base, d1 = tmem_base + kAccCols;
    for (int it = 0; tm.at(tq.pop(), t); ++it) {
      const int npad = (__shfl_sync(0xffffffffu, p.wl.run_n[t.run], 0) + 15) & ~15;
      CAEE_DEV_ASSERT(npad >= 16 && npad <= kRunTokens && p.wl.run_hrow[t.run] + npad <= p.wl.hrow_cap);
      const uint32_t idesc = (1u << 4) | ((uint32_t)(npad >> 3) << 17) | ((uint32_t)(kTileRows >> 4) << 24);   // fp16 x fp16 -> fp32
      const int nkb = t.phase == 1 ? p.KB1 : p.KB2;
      const uint32_t sub_bytes = (uint32_t)npad * 128u;       // one 64-k image of the run inside a token stage
      WAIT_T(w_a, mbar_wait(tempty, (it & 1) ^ 1));
      tc_fence_after();
      if constexpr (kSubK == 128) {
        for (int s = 0; s < nkb; ++s) {
          WAIT_T(w_b, mbar_wait(cfull0 + 8 * cs, cph));
          WAIT_T(w_c, mbar_wait(kfull0 + 8 * ks, kph));
          tc_fence_after();
          const uint32_t a0 = tmem_base + kACol0 + cs * kAStageCols, a1 = a0 + kAStageCols / 2;
          const uint64_t b0 = make_desc_sw128(smem_base + ks * kTokBytes), b1 = make_desc_sw128(smem_base + ks * kTokBytes + sub_bytes);
          if (elect_one()) {
            if (s == 0) {
              umma_f16_ts<false>(d0, a0, b0, idesc);
              umma_f16_ts<false>(d1, a1, b0, idesc);
            } else {
              umma_f16_ts<true>(d0, a0, b0, idesc);
              umma_f16_ts<true>(d1, a1, b0, idesc);
            }
#pragma unroll
            for (int k16 = 1; k16 < kKRaw / 16; ++k16) {   // per 16-k step: weights +8 TMEM columns, tokens +32 B (>> 4) inside a 64-k image
              const uint64_t b = (k16 < 4 ? b0 : b1) + (uint64_t)((k16 & 3) * 2);
              umma_f16_ts<true>(d0, a0 + k16 * 8, b, idesc);
              umma_f16_ts<true>(d1, a1 + k16 * 8, b, idesc);
            }
            tc_commit(cempty0 + 8 * cs);
            tc_commit(kempty0 + 8 * ks);
            if (s == nkb - 1) tc_commit(tfull);
          }
          __syncwarp();
          if (++cs == kAStagesT) { cs = 0; cph ^= 1; }
          if (++ks == kTokStages) { ks = 0; kph ^= 1; }
        }
      } else {
        // 64-k stages on both rings: 2 nkb hand-overs of 8 MMAs each
        for (int s = 0; s < 2 * nkb; ++s) {
          WAIT_T(w_b, mbar_wait(cfull0 + 8 * cs, cph));
          WAIT_T(w_c, mbar_wait(kfull0 + 8 * ks, kph));
          tc_fence_after();
          const uint32_t a0 = tmem_base + kACol0 + cs * kAStageCols, a1 = a0 + kAStageCols / 2;
          const uint64_t b0 = make_desc_sw128(smem_base + ks * kTokBytes);
          if (elect_one()) {
            if (s == 0) {
              umma_f16_ts<false>(d0, a0, b0, idesc);
              umma_f16_ts<false>(d1, a1, b0, idesc);
            } else {
              umma_f16_ts<true>(d0, a0, b0, idesc);
              umma_f16_ts<true>(d1, a1, b0, idesc);
            }
#pragma unroll
            for (int k16 = 1; k16 < 4; ++k16) {
              umma_f16_ts<true>(d0, a0 + k16 * 8, b0 + (uint64_t)(k16 * 2), idesc);
              umma_f16_ts<true>(d1, a1 + k16 * 8, b0 + (uint64_t)(k16 * 2), idesc);
            }
            tc_commit(cempty0 + 8 * cs);
            tc_commit(kempty0 + 8 * ks);
            if (s == 2 * nkb - 1) tc_commit(tfull);
          }
          __syncwarp();
          if (++cs == kAStagesT) { cs = 0; cph ^= 1; }
          if (++ks == kTokStages) { ks = 0; kph ^= 1; }
        }
      }
    }
  } else if (warp == 2) {
    // ===== token-operand loader: ONE bulk copy per token stage (kSubK k: one or two consecutive 64-k images) from the run's stage images
    if (lane == 0) {
      int stage = 0, ph = 0;
      while (tm.at(tq.pop1(), t)) {
        const int npad = (p.wl.run_n[t.run] + 15) & ~15;
        const int nsub = (t.phase == 1 ? p.KB1 : p.KB2) * (kKRaw / kSubK);
        const size_t row_bytes = (size_t)(t.phase == 1 ? p.H : p.I) * 2;
        const uint32_t stage_bytes = (uint32_t)npad * (uint32_t)(kSubK * 2);   // kSubK / 64 consecutive 64-k images of the run: one copy
        const uint8_t* src = (t.phase == 1 ? p.xg : p.hbuf) + (size_t)p.wl.run_hrow[t.run] * row_bytes;
        if (t.phase == 2) {
          const int* flag = p.wl.ready + t.run;
          while (ld_acquire(flag) < p.P1) __nanosleep(64);
          asm volatile("fence.proxy.async;" ::: "memory");
        }
        for (int s = 0; s < nsub; ++s) {
          mbar_wait(kempty0 + 8 * stage, ph ^ 1);
          mbar_arrive_expect_tx(kfull0 + 8 * stage, stage_bytes);
          bulk_g2s(smem_base + stage * kTokBytes, src + (size_t)s * stage_bytes, stage_bytes, kfull0 + 8 * stage);
          if (++stage == kTokStages) { stage = 0; ph ^= 1; }
        }
      }
    }
  } else if (warp == 3) {
    // spare warp
  } else if (warp < 8 || warp >= 16) {
    // ===== epilogue (warps 4-7 and 16-19): two warps per TMEM lane quadrant q = warp % 4, each one half of the
    // token columns (as in expert_fp8_wide.cu)
    const int q = warp & 3, eh = warp >= 16;
    for (int it = 0; tm.at(tq.pop(), t); ++it) {
      const int n = p.wl.run_n[t.run], start = p.wl.run_start[t.run];
      const int npad = (n + 15) & ~15;
      const int half = (((npad >> 4) + 1) >> 1) << 4;
      const int c_lo = eh ? half : 0, c_hi = eh ? n : min(half, n);
      int dst_l[kRunTokens / 64];
      if (t.phase == 2) {
#pragma unroll
        for (int i = 0; i < kRunTokens / 64; ++i) {
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
              const float hv = fminf(fmaxf(__fdividef(gv, 1.0f + __expf(-gv)) * uv, -65504.f), 65504.f);
              const int cc = c + j;
              *reinterpret_cast<uint16_t*>(hrun + cc * 128 + ((chunk ^ (cc & 7)) << 4)) = __half_as_ushort(__float2half_rn(hv));
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
          for (int i = 0; i < kRunTokens / 64; ++i)
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
      if (lane == 0) mbar_arrive(tempty);
      if (t.phase == 1) {
        asm volatile("fence.proxy.async;" ::: "memory");
        __threadfence();
        asm volatile("bar.sync 1, 256;" ::: "memory");
        if (threadIdx.x == 128) atomicAdd(p.wl.ready + t.run, 1);
      }
    }
  } else {
    // ===== converters (warps 8-15): thread = weight row `row` of tile half th; per 64-k stage its 64 codes
    // (4 chunks of 16, 128 bytes apart in the packed stage) -> fp16 x block scale -> 32 TMEM columns
    const int th = (warp - 8) >> 2, q = warp & 3;
    const int row = q * 32 + lane;
    const int row_off = th * kATileBytes + (row >> 3) * 1024 + (row & 7) * 16;   // this row's first chunk in a packed stage
    const uint32_t trow = tmem_base + ((uint32_t)(q * 32) << 16) + kACol0 + th * (kAStageCols / 2);
    int cs = 0, cph = 0, rs = 0, rph = 0;
    while (tm.at(tq.pop(), t)) {
      const int nkb = t.phase == 1 ? p.KB1 : p.KB2;
      const uint8_t* img = p.packed[p.wl.run_expert[t.run]];
      const float* tab = reinterpret_cast<const float*>(img + p.sc_off);
      const float* wsc = t.phase == 1 ? tab + (size_t)t.sub * p.KB1 * 2 : tab + p.t2_off + (size_t)t.sub * p.KB2 * 2;
      const float nrm = __ldg(reinterpret_cast<const float*>(img + p.norm_off));
      // the tile's block scales of this half, fetched once: lane l keeps those of k blocks l, l + 32
      float sc[kMaxKb / 32];
#pragma unroll
      for (int j = 0; j < kMaxKb / 32; ++j) {
        const int kbj = lane + 32 * j;
        sc[j] = kbj < nkb ? __ldg(wsc + 2 * kbj + th) * nrm : 0.f;
      }
      for (int kb = 0; kb < nkb; ++kb) {
        float s0 = 0.f;
#pragma unroll
        for (int j = 0; j < kMaxKb / 32; ++j)
          if ((kb >> 5) == j) s0 = sc[j];
        const __half2 w2 = __float2half2_rn(__shfl_sync(0xffffffffu, s0, kb & 31));
        WAIT_T(w_c, mbar_wait(rfull0 + 8 * rs, rph));          // the stage's codes have landed (bulk copy)
        const uint8_t* raw = smem + kRawOff + rs * kAStageBytes + row_off;
        if constexpr (kSubK == 128) {
          WAIT_T(w_a, mbar_wait(cempty0 + 8 * cs, cph ^ 1));     // the MMAs that read this A stage are done
          tc_fence_after();
#pragma unroll
          for (int hh = 0; hh < 2; ++hh) {
            uint32_t o[32];
#pragma unroll
            for (int i = 0; i < 4; ++i) widen16_ts(*reinterpret_cast<const uint4*>(raw + hh * 512 + i * 128), w2, o + 8 * i);
            tmem_st32(trow + cs * kAStageCols + hh * 32, o);
          }
          __syncwarp();
          if (lane == 0) mbar_arrive(rempty0 + 8 * rs);      // this warp has read its rows of the stage
          WAIT_T(w_b, tmem_st_wait());
          tc_fence_before();
          __syncwarp();
          if (lane == 0) mbar_arrive(cfull0 + 8 * cs);
          if (++cs == kAStagesT) { cs = 0; cph ^= 1; }
        } else {
          // 64-k A stages: each half of the raw stage is its own hand-over
#pragma unroll
          for (int hh = 0; hh < 2; ++hh) {
            uint32_t o[32];
#pragma unroll
            for (int i = 0; i < 4; ++i) widen16_ts(*reinterpret_cast<const uint4*>(raw + hh * 512 + i * 128), w2, o + 8 * i);
            if (hh == 1) {
              __syncwarp();
              if (lane == 0) mbar_arrive(rempty0 + 8 * rs);    // both halves of this warp's rows are in registers
            }
            WAIT_T(w_a, mbar_wait(cempty0 + 8 * cs, cph ^ 1));
            tc_fence_after();
            tmem_st32(trow + cs * kAStageCols, o);
            WAIT_T(w_b, tmem_st_wait());
            tc_fence_before();
            __syncwarp();
            if (lane == 0) mbar_arrive(cfull0 + 8 * cs);
            if (++cs == kAStagesT) { cs = 0; cph ^= 1; }
          }
        }
        if (++rs == kRawStages) { rs = 0; rph ^= 1; }
      }
    }
  }

#ifdef CAEE_WIDE_STATS
  if (lane == 0 && (blockIdx.x == 0 || blockIdx.x == 101) && (warp == 1 || warp == 8 || warp == 4))
    printf("ts cta %d warp %d: total %lld  wait a %lld b %lld c %lld d %lld\n", blockIdx.x, warp, clock64() - t_start, w_a, w_b, w_c, w_d);
#endif
  tc_fence_before();
  __syncthreads();
  if (warp == 2) {
    tc_fence_after();
    asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;" ::"r"(tmem_base), "n"(kTmemCols));
  }
}

}  // namespace

// runs [run_begin, run_begin + run_count) (run_count < 0: every run of the work list), tile tickets from
// wl.sched[ticket].  Runs hold up to wl.run_cap = CAEE_RUN_TOKENS_TS (192) or CAEE_RUN_TOKENS (128) tokens; x images by
// caee_launch_fp8_wide_prepare.
void caee_launch_expert_fp8_ts(caee_ctx* c, int T, int run_begin, int run_count, int ticket, cudaStream_t st) {
  (void)T;
  ++c->n_launches;
  const caee_layer_desc& d = c->d;
  TsParams p;
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
  if (c->wl.run_cap > CAEE_RUN_TOKENS) {
    if (!(c->attr_done & 32u)) {
      cudaFuncSetAttribute(k_expert_fp8_ts<CAEE_RUN_TOKENS_TS>, cudaFuncAttributeMaxDynamicSharedMemorySize, TsCfg<CAEE_RUN_TOKENS_TS>::kSmemBytes + 1024);
      c->attr_done |= 32u;
    }
    k_expert_fp8_ts<CAEE_RUN_TOKENS_TS><<<c->num_sms, kThreads, TsCfg<CAEE_RUN_TOKENS_TS>::kSmemBytes + 1024, st>>>(p);
    return;
  }
  if (!(c->attr_done & 16u)) {
    cudaFuncSetAttribute(k_expert_fp8_ts<CAEE_RUN_TOKENS>, cudaFuncAttributeMaxDynamicSharedMemorySize, TsCfg<CAEE_RUN_TOKENS>::kSmemBytes + 1024);
    c->attr_done |= 16u;
  }
  k_expert_fp8_ts<CAEE_RUN_TOKENS><<<c->num_sms, kThreads, TsCfg<CAEE_RUN_TOKENS>::kSmemBytes + 1024, st>>>(p);
}
