// expert_fp8.cu — S7 grouped SwiGLU expert FFN for FP8-E4M3 weights with 128x128 block scales
// (BASELINE.json config 4) on sm_100a: the weight bytes go from HBM to the tensor cores
// untouched.
//
// Design.  At decode the bound is HBM bandwidth (Fig. 1), so the e4m3 codes are
// streamed exactly once by the bulk async-copy engine into a shared-memory ring and fed to
// tcgen05.mma kind::f8f6f4 as they are — no widening pass through shared memory (a converter
// design spends 5x the HBM byte rate in shared-memory traffic and cannot keep up).  The tensor
// cores need both operands in a narrow format, and rounding the bf16 activations to e4m3
// would miss the 5e-2 x RMS tolerance, so each activation is split into TWO e4m3 terms,
//     a / s = hi + lo,   hi = e4m3(a / s),   lo = e4m3(a / s - hi),
// with one fp32 scale s = amax/448 per (token, 128-wide k block): 2^-8 relative error per
// element, about bf16's own rounding.  Both terms accumulate into the same TMEM accumulator
// (two MMAs per weight tile and k-step; the tensor pipe is far from busy at decode).
// Block scales: a stage is one 128-k block of a 128-row tile pair, i.e. ONE weight scale per
// accumulator, so the MMA warp gives every k block a fresh TMEM accumulator (double buffered)
// and the epilogue warps promote it into fp32 registers:
//     acc[row, tok] += D_kb[row, tok] * w_scale[tile half, kb] * a_scale[tok, kb].
// x is split once per step (k_act_split); h is split by the phase-1 epilogue that produces it.
//
// Layout.  caee_set_weights(pack=1) rewrites every expert into 32 KB stage images: two 128-row x
// 128-k e4m3 tiles in the UMMA canonical K-major no-swizzle order (8 rows x 16 B core matrices;
// LBO 128 B, SBO 1024 B), phase 1 = [gate tile | up tile] of the same 128 features, phase 2 =
// down rows [+0..127 | +128..255]; then the fp32 block-scale table, [tile][kb][half].
//
// Roles (384 threads, 1 CTA per SM): warp 0 = weight producer (bulk copies), warp 1 = MMA
// issuer, warp 2 = token-operand loader (TMA row gathers of the hi/lo rows), warps 4-11 =
// epilogue (two warps per TMEM lane quadrant, each half of the token columns).  Tiles are
// claimed by atomic ticket, phase-1 tickets first (see umma_common.cuh).
#include <cstring>

#include "umma_common.cuh"
#include "act_split_dev.cuh"

namespace {

using namespace caee_umma;

constexpr int kThreads = 384;
constexpr int kKBlock = 128;      // k elements per stage = one block-scale block
constexpr int kEpiWarps = 8;

struct Fp8Params {
  caee_worklist wl;
  uint8_t* const* packed;   // [E+S] stage images + scale table
  const uint8_t* xq_hi;     // [T,H] e4m3
  const uint8_t* xq_lo;     // [T,H]
  const float* xs;          // [T,H/128]
  uint8_t* hq_hi;           // [rows,I]
  uint8_t* hq_lo;
  float* hs;                // [rows,I/128]
  float* obuf;              // [T*(k+S),H]
  int H, I;
  int P1, P2, KB1, KB2;     // tiles per run and 128-k stages per tile, per phase
  int n_stages, stage_bytes, b_term_bytes;
  int run_begin, run_count, ticket;
  int sc_off;               // byte offset of the scale table in a packed image
  int t2_off;               // float offset of its phase-2 part
  // token operand by TMA row gather (tile::gather4, 128 B rows, 128 B swizzle): 2D maps over the
  // [hi rows | lo rows] x k byte arrays of x and of h; lo row = hi row + lo_row_*
  CUtensorMap tm_x, tm_h;
  int lo_row_x, lo_row_h;
  KSplit ksp;               // split k range of phase-1 tiles in steps of a few tokens (umma_common.cuh)
};

__device__ __forceinline__ uint16_t cvt_e4m3x2(float a, float b) { return caee_cvt_e4m3x2(a, b); }
__device__ __forceinline__ float2 e4m3x2_to_float2(uint16_t v) { return caee_e4m3x2_to_float2(v); }

// Once per step: x[T,H] bf16 -> hi/lo e4m3 terms and the (token, 128-block) scales (act_split_dev.cuh).
// One warp per block of 128 elements.  (Steps of <= 16 tokens: the decision kernel does this itself.)
__global__ void __launch_bounds__(256) k_act_split(const __nv_bfloat16* __restrict__ x, uint8_t* __restrict__ hi,
                                                   uint8_t* __restrict__ lo, float* __restrict__ scale, size_t n_blocks) {
  const size_t b = (size_t)blockIdx.x * 8 + (threadIdx.x >> 5);
  if (b >= n_blocks) return;
  caee_act_split_block(x, hi, lo, scale, b, threadIdx.x & 31);
}

// One thread per 16 codes: raw row-major [rows, cols] e4m3 -> stage images.
// which: 0 gate, 1 up (phase-1 region), 2 down (phase-2 region).
__global__ void __launch_bounds__(256) k_pack_e4m3(const uint8_t* __restrict__ src, uint8_t* __restrict__ dst, int rows,
                                                   int cols, int which, size_t region_off) {
  const size_t chunk = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
  const int cpr = cols / 16;
  if (chunk >= (size_t)rows * cpr) return;
  const int r = (int)(chunk / cpr), k0 = (int)(chunk % cpr) * 16;
  const int kb = k0 / kKBlock, kk = k0 % kKBlock, nkb = cols / kKBlock;
  int tile, half;
  const int rr = r % kTileRows;
  if (which < 2) { tile = r / kTileRows; half = which; }
  else { tile = r / (2 * kTileRows); half = (r / kTileRows) & 1; }
  const size_t stage = (size_t)tile * nkb + kb;
  const size_t in_stage = (size_t)half * kATileBytes + (rr / 8) * 1024 + (kk / 16) * 128 + (rr % 8) * 16;
  const uint4 v = *reinterpret_cast<const uint4*>(src + (size_t)r * cols + k0);
  *reinterpret_cast<uint4*>(dst + region_off + stage * kAStageBytes + in_stage) = v;
}

// Block-scale table of one expert: tab[(tile * KS + kb) * 2 + half], phase-1 tiles first.
//   phase 1, tile ft:  halves = gate rows / up rows of feature block ft   (scale row ft of each)
//   phase 2, tile op:  halves = down rows 256 op + [0,128) / + [128,256)  (scale rows 2 op, 2 op + 1)
__global__ void k_scale_table(const float* __restrict__ sg, const float* __restrict__ su, const float* __restrict__ sd,
                              float* __restrict__ tab, int P1, int P2, int KS1, int KS2) {
  const int n1 = P1 * KS1 * 2, n2 = P2 * KS2 * 2;
  for (int i = blockIdx.x * blockDim.x + threadIdx.x; i < n1 + n2; i += gridDim.x * blockDim.x) {
    if (i < n1) {
      const int half = i & 1, kb = (i >> 1) % KS1, ft = (i >> 1) / KS1;
      tab[i] = (half ? su : sg)[(size_t)ft * KS1 + kb];
    } else {
      const int j = i - n1, half = j & 1, kb = (j >> 1) % KS2, op = (j >> 1) / KS2;
      tab[i] = sd[(size_t)(2 * op + half) * KS2 + kb];
    }
  }
}

// Per-expert power of two 2^J with max |scale| 2^J in [64, 128): the converter kernels
// (expert_fp8_ts.cu, expert_fp8_wide.cu) fold scale 2^J into fp16 weights (|code| <= 448, so products stay below
// 65504) and multiplies its accumulators by 2^-J.  norm[0] = 2^J, norm[1] = 2^-J.
__global__ void __launch_bounds__(256) k_scale_norm(const float* __restrict__ tab, int n, float* __restrict__ norm) {
  __shared__ float red[8];
  float m = 0.f;
  for (int i = threadIdx.x; i < n; i += 256) {
    const float v = fabsf(tab[i]);
    if (v <= 3.0e38f) m = fmaxf(m, v);   // skips inf / nan
  }
#pragma unroll
  for (int o = 16; o; o >>= 1) m = fmaxf(m, __shfl_xor_sync(0xffffffffu, m, o));
  if ((threadIdx.x & 31) == 0) red[threadIdx.x >> 5] = m;
  __syncthreads();
  if (threadIdx.x == 0) {
    for (int i = 1; i < 8; ++i) m = fmaxf(m, red[i]);
    int ex = 7;
    if (m > 0.f) frexpf(m, &ex);          // m = f 2^ex, f in [0.5, 1)
    int J = 7 - ex;
    J = max(-100, min(100, J));
    norm[0] = ldexpf(1.0f, J);
    norm[1] = ldexpf(1.0f, -J);
  }
}

// ------------------------------------------------------------------ the kernel, part 1: roles 0-3
__global__ void __launch_bounds__(kThreads, 1) k_expert_fp8(const __grid_constant__ Fp8Params p);

#ifdef CAEE_TILE_TRACE
// tuning aid (not in the product build): per tile {sm, ticket, claim, first copy issued, last copy issued, epilogue done} in ns
__device__ long long g_tile_trace[4096][6];
__device__ __forceinline__ long long gtime() { long long t; asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(t)); return t; }
__device__ __forceinline__ int smid() { int s; asm volatile("mov.u32 %0, %%smid;" : "=r"(s)); return s; }
#endif

// Per-tile epilogue body for CT token columns per warp (defined below).
template <int CT>
__device__ __forceinline__ void fp8_epilogue_tile(const Fp8Params& p, const Tile& t, uint32_t tmem_base, uint32_t tfull0,
                                                  uint32_t tempty0, int& acc_it, int& p1_it, float (*amax_s)[kTileRows], int q,
                                                  int hf, int lane, int KS);

__global__ void __launch_bounds__(kThreads, 1) k_expert_fp8(const __grid_constant__ Fp8Params p) {
  extern __shared__ __align__(1024) uint8_t smem_raw[];
  uint8_t* smem = reinterpret_cast<uint8_t*>((reinterpret_cast<uintptr_t>(smem_raw) + 1023) & ~(uintptr_t)1023);
  __shared__ __align__(8) uint64_t bars[2 * kMaxStages + 4 + 2 * kQueue];
  __shared__ uint32_t tmem_base_s;
  __shared__ int tq_slots[kQueue];
  __shared__ float amax_s[3][kTileRows];   // per-token |h| maxima of a phase-1 tile (3 buffers in rotation)

  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const uint32_t smem_base = smem_u32(smem);
  const uint32_t full0 = smem_u32(&bars[0]), empty0 = smem_u32(&bars[kMaxStages]);
  const uint32_t tfull0 = smem_u32(&bars[2 * kMaxStages]), tempty0 = smem_u32(&bars[2 * kMaxStages + 2]);
  const uint32_t qfull0 = smem_u32(&bars[2 * kMaxStages + 4]), qempty0 = smem_u32(&bars[2 * kMaxStages + 4 + kQueue]);

  if (threadIdx.x == 0) {
    for (int s = 0; s < p.n_stages; ++s) {
      mbar_init(full0 + 8 * s, 2);   // expect_tx arrives of the weight producer and of the token-operand loader
      mbar_init(empty0 + 8 * s, 1);  // tcgen05.commit
    }
    for (int a = 0; a < 2; ++a) {
      mbar_init(tfull0 + 8 * a, 1);           // tcgen05.commit
      mbar_init(tempty0 + 8 * a, kEpiWarps);  // one lane of each epilogue warp
    }
    for (int q = 0; q < kQueue; ++q) {
      mbar_init(qfull0 + 8 * q, 1);               // producer
      mbar_init(qempty0 + 8 * q, 2 + kEpiWarps);  // MMA warp + loader warp + epilogue warps
    }
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
  }
  for (int i = threadIdx.x; i < 3 * kTileRows; i += kThreads) (&amax_s[0][0])[i] = 0.f;
  if (warp == 2) {
    asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], %1;" ::"r"(smem_u32(&tmem_base_s)),
                 "n"(kTmemCols));
    asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;");
  }
  tc_fence_before();
  __syncthreads();
  tc_fence_after();
  const uint32_t tmem_base = tmem_base_s;
  // everything above touched only shared memory and TMEM: with a programmatic dependent launch it
  // overlaps the decision kernel's tail; the work list exists from here on
  griddep_wait();
  griddep_launch();
  const int n_runs = p.run_count >= 0 ? p.run_count : p.wl.meta[1];
  const int KS = (p.ksp.ks > 1 && n_runs * p.P1 <= p.ksp.tile_cap) ? p.ksp.ks : 1;
  const TileMap tm{n_runs, p.run_begin, p.P1, p.P2, KS};
  const int KB1s = p.KB1 / KS;             // 128-k stages of one phase-1 (sub-)tile
  TileQueue tq{qfull0, qempty0, tq_slots, 0, 0};
  Tile t;

  if (warp == 0) {
    // ===== weight producer: claims tiles; one 32 KB bulk copy per 128-k stage from the packed image
    if (lane == 0) {
      int stage = 0, ph = 0, q = 0, qph = 0;
      const uint64_t pol = l2_evict_first_policy();
      // where a tile's stages start in its expert's packed image, and how many there are
      auto resolve = [&](const Tile& tt, const uint8_t*& src, int& nkb) {
        const int e = p.wl.run_expert[tt.run];
        nkb = tt.phase == 1 ? KB1s : p.KB2;
        src = p.packed[e] + (tt.phase == 1 ? (size_t)tt.sub * p.KB1 + (size_t)tt.kq * KB1s : (size_t)p.P1 * p.KB1 + (size_t)tt.sub * p.KB2) * kAStageBytes;
      };
      // The next tile's ticket (an atomic round trip) and its image pointer (two dependent loads) are
      // fetched while the current tile's copies are being issued: claimed and resolved at the tile
      // boundary they left the copy engine idle for ~1.2 us per tile.  (Tickets still come in
      // increasing order per CTA; every CTA ends on a ticket beyond the last tile.)  The first tile of CTA b is tile b:
      // no atomic round trip before the first weight byte is requested; the counter hands out tiles gridDim.x, ...
      int nxt = (int)blockIdx.x;
      Tile tn;
      const uint8_t* srcn = nullptr;
      int nkbn = 0;
      bool vn = tm.at(nxt, tn);
      if (vn) resolve(tn, srcn, nkbn);
      for (;;) {
        const int i = nxt, nkb = nkbn;
        const uint8_t* src = srcn;
        mbar_wait(qempty0 + 8 * q, qph ^ 1);
        tq_slots[q] = i;
        mbar_arrive(qfull0 + 8 * q);
        if (++q == kQueue) { q = 0; qph ^= 1; }
        if (!vn) break;
#ifdef CAEE_TILE_TRACE
        if (i < 4096) { g_tile_trace[i][0] = smid(); g_tile_trace[i][1] = i; g_tile_trace[i][2] = gtime(); }
#endif
        nxt = (int)gridDim.x + atomicAdd(p.wl.sched + p.ticket, 1);
        for (int kb = 0; kb < nkb; ++kb) {
          mbar_wait(empty0 + 8 * stage, ph ^ 1);
          mbar_arrive_expect_tx(full0 + 8 * stage, kAStageBytes);
          bulk_g2s_stream(smem_base + stage * p.stage_bytes, src + (size_t)kb * kAStageBytes, kAStageBytes, full0 + 8 * stage, pol);
#ifdef CAEE_TILE_TRACE
          if (i < 4096 && kb == 0) g_tile_trace[i][3] = gtime();
          if (i < 4096 && kb == nkb - 1) g_tile_trace[i][4] = gtime();
#endif
          if (++stage == p.n_stages) { stage = 0; ph ^= 1; }
          if (kb == (nkb >> 1)) {
            vn = tm.at(nxt, tn);
            if (vn) resolve(tn, srcn, nkbn);
          }
        }
      }
    }
  } else if (warp == 1) {
    // ===== MMA issuer: every 128-k stage gets a fresh TMEM accumulator pair (block-scale promotion).
    // The whole warp runs the loop (uniform control flow); one elected lane issues.
    int stage = 0, ph = 0, acc_it = 0;
    while (tm.at(tq.pop(), t)) {
      const int nkb = t.phase == 1 ? KB1s : p.KB2;
      const int npad = (__shfl_sync(0xffffffffu, p.wl.run_n[t.run], 0) + 15) & ~15;
      // up to 64 tokens the lo rows follow the hi rows and ONE MMA of N = 2 npad takes both terms
      // (hi and lo partial sums in separate columns, added by the epilogue): the weight tile is
      // read from shared memory once per k-step.  Wider runs add both terms into the same columns.
      const bool cat = npad <= 64;
      const uint32_t idesc = make_idesc(cat ? 2 * npad : npad, false);   // e4m3 x e4m3 (format 0), fp32 accumulate
      for (int kb = 0; kb < nkb; ++kb, ++acc_it) {
        const int as = acc_it & 1;
        mbar_wait(tempty0 + 8 * as, ((acc_it >> 1) & 1) ^ 1);
        mbar_wait(full0 + 8 * stage, ph);
        tc_fence_after();
        const uint32_t d0 = tmem_base + as * 256, d1 = d0 + 128;
        const uint32_t a_addr = smem_base + stage * p.stage_bytes;
        const uint64_t a0 = make_desc(a_addr), a1 = make_desc(a_addr + kATileBytes);
        const uint64_t bh = make_desc_sw128(a_addr + kAStageBytes), bl = make_desc_sw128(a_addr + kAStageBytes + p.b_term_bytes);
        if (elect_one()) {
          if (cat) {
            umma_f8_imm<false>(d0, a0, bh, idesc);
            umma_f8_imm<false>(d1, a1, bh, idesc);
#pragma unroll
            for (int ks = 1; ks < kKBlock / 32; ++ks) {     // per 32-element k-step: weights +256 B, tokens +32 B (>> 4)
              umma_f8_imm<true>(d0, a0 + (uint64_t)(ks * 16), bh + (uint64_t)(ks * 2), idesc);
              umma_f8_imm<true>(d1, a1 + (uint64_t)(ks * 16), bh + (uint64_t)(ks * 2), idesc);
            }
          } else {
            umma_f8_imm<false>(d0, a0, bh, idesc);
            umma_f8_imm<true>(d0, a0, bl, idesc);
            umma_f8_imm<false>(d1, a1, bh, idesc);
            umma_f8_imm<true>(d1, a1, bl, idesc);
#pragma unroll
            for (int ks = 1; ks < kKBlock / 32; ++ks) {
              const uint64_t o = (uint64_t)(ks * 16), ob = (uint64_t)(ks * 2);
              umma_f8_imm<true>(d0, a0 + o, bh + ob, idesc);
              umma_f8_imm<true>(d0, a0 + o, bl + ob, idesc);
              umma_f8_imm<true>(d1, a1 + o, bh + ob, idesc);
              umma_f8_imm<true>(d1, a1 + o, bl + ob, idesc);
            }
          }
          tc_commit(empty0 + 8 * stage);
          tc_commit(tfull0 + 8 * as);
        }
        __syncwarp();
        if (++stage == p.n_stages) { stage = 0; ph ^= 1; }
      }
    }
  } else if (warp == 2) {
    // ===== token-operand loader: TMA row gathers (4 rows x 128 B per instruction) of the hi and lo
    // e4m3 rows of x (phase 1) or h (phase 2) into 128-byte-swizzled 8-row atoms; lane l owns rows
    // 4l..4l+3 of the run, padding rows come back as zeros
    int stage = 0, ph = 0;
    while (tm.at(tq.pop(), t)) {
      const int n = p.wl.run_n[t.run], start = p.wl.run_start[t.run];
      const int npad = (n + 15) & ~15;
      const int nkb = t.phase == 1 ? KB1s : p.KB2, kb0 = t.kq * KB1s;     // kq = 0 in phase 2
      const uint32_t lo_smem = npad <= 64 ? (uint32_t)npad * kKBlock : (uint32_t)p.b_term_bytes;   // see the MMA warp
      const CUtensorMap* tmap = t.phase == 1 ? &p.tm_x : &p.tm_h;
      const int lo_row = t.phase == 1 ? p.lo_row_x : p.lo_row_h;
      int rh[4], rl[4];
#pragma unroll
      for (int i = 0; i < 4; ++i) {
        const int row = lane * 4 + i;
        rh[i] = kOobRow; rl[i] = kOobRow;
        if (row < n) {
          rh[i] = t.phase == 1 ? p.wl.ent_tok[start + row] : p.wl.run_hrow[t.run] + row;
          rl[i] = rh[i] + lo_row;
        }
      }
      if (t.phase == 2) {
        // h of this run is complete once all P1 gate/up tiles have published it (generic-proxy
        // stores of other SMs, read here through the async proxy)
        if (lane == 0) {
          const int* flag = p.wl.ready + t.run;
          while (ld_acquire(flag) < p.P1) __nanosleep(64);
        }
        __syncwarp();
        asm volatile("fence.proxy.async;" ::: "memory");
      }
      CAEE_DEV_ASSERT(n >= 1 && n <= p.wl.run_cap && start >= 0 && start + n <= p.wl.ent_cap && p.wl.run_hrow[t.run] + npad <= p.wl.hrow_cap);
      const bool mine = lane * 4 < npad;
      for (int kb = 0; kb < nkb; ++kb) {
        mbar_wait(empty0 + 8 * stage, ph ^ 1);
        const uint32_t b_addr = smem_base + stage * p.stage_bytes + kAStageBytes;
        if (lane == 0) mbar_arrive_expect_tx(full0 + 8 * stage, 2u * npad * kKBlock);
        __syncwarp();
        if (mine) {
          tma_gather4(b_addr + lane * 512, tmap, full0 + 8 * stage, (kb0 + kb) * kKBlock, rh[0], rh[1], rh[2], rh[3]);
          tma_gather4(b_addr + lo_smem + lane * 512, tmap, full0 + 8 * stage, (kb0 + kb) * kKBlock, rl[0], rl[1], rl[2], rl[3]);
        }
        if (++stage == p.n_stages) { stage = 0; ph ^= 1; }
      }
    }
  } else if (warp == 3) {
    // ===== reducer (only in steps that split their phase-1 tiles, KSplit): finishes tiles whose ks
    // partial sums are complete: h = silu(gate) * up, its (token, 128-feature block) scale and two e4m3
    // terms — the arithmetic of the unsplit epilogue below; lane l holds features 4 l .. 4 l + 3
    if (KS > 1) {
      const int n_tiles = n_runs * p.P1;
      for (int first = 1;; first = 0) {
        int j = (int)blockIdx.x;                                  // the first tile of CTA b's reducer is tile b
        if (!first) {
          if (lane == 0) j = (int)gridDim.x + atomicAdd(p.wl.sched + p.ksp.rticket, 1);
          j = __shfl_sync(0xffffffffu, j, 0);
        }
        if (j >= n_tiles) break;
        const int run = p.run_begin + j / p.P1, ft = j % p.P1;
        const int n = p.wl.run_n[run], hrow = p.wl.run_hrow[run];
        if (lane == 0) {
          while (ld_acquire(p.ksp.cnt + j) < KS) __nanosleep(100);
          p.ksp.cnt[j] = 0;                     // every sub-tile has arrived: ready for the next step
        }
        __syncwarp();
        const float* part = p.ksp.part + (size_t)j * KS * (2 * kKSplitCols * kTileRows) + 4 * lane;
        for (int c = 0; c < n; ++c) {
          float4 g = make_float4(0.f, 0.f, 0.f, 0.f), u = g;
          for (int kq = 0; kq < KS; ++kq) {
            const float4 a = __ldcg(reinterpret_cast<const float4*>(part + (kq * 2 * kKSplitCols + c) * kTileRows));
            const float4 b = __ldcg(reinterpret_cast<const float4*>(part + (kq * 2 * kKSplitCols + kKSplitCols + c) * kTileRows));
            g.x += a.x; g.y += a.y; g.z += a.z; g.w += a.w;
            u.x += b.x; u.y += b.y; u.z += b.z; u.w += b.w;
          }
          const float h0 = g.x / (1.0f + __expf(-g.x)) * u.x, h1 = g.y / (1.0f + __expf(-g.y)) * u.y;
          const float h2 = g.z / (1.0f + __expf(-g.z)) * u.z, h3 = g.w / (1.0f + __expf(-g.w)) * u.w;
          float m = fmaxf(fmaxf(fabsf(h0), fabsf(h1)), fmaxf(fabsf(h2), fabsf(h3)));
#pragma unroll
          for (int o = 16; o; o >>= 1) m = fmaxf(m, __shfl_xor_sync(0xffffffffu, m, o));
          const float sc = m > 0.f ? m * (1.0f / 448.0f) : 1.0f;
          const float v0 = h0 / sc, v1 = h1 / sc, v2 = h2 / sc, v3 = h3 / sc;
          const uint16_t hi01 = cvt_e4m3x2(v0, v1), hi23 = cvt_e4m3x2(v2, v3);
          const float2 f01 = e4m3x2_to_float2(hi01), f23 = e4m3x2_to_float2(hi23);
          const uint16_t lo01 = cvt_e4m3x2(v0 - f01.x, v1 - f01.y), lo23 = cvt_e4m3x2(v2 - f23.x, v3 - f23.y);
          const size_t off = (size_t)(hrow + c) * p.I + ft * kTileRows + 4 * lane;
          *reinterpret_cast<uint32_t*>(p.hq_hi + off) = (uint32_t)hi01 | ((uint32_t)hi23 << 16);
          *reinterpret_cast<uint32_t*>(p.hq_lo + off) = (uint32_t)lo01 | ((uint32_t)lo23 << 16);
          if (lane == 0) p.hs[(size_t)(hrow + c) * p.KB2 + ft] = sc;
        }
        // publish the tile's slice of h (read through the async proxy by other SMs' TMA gathers)
        asm volatile("fence.proxy.async;" ::: "memory");
        __threadfence();
        __syncwarp();
        if (lane == 0) atomicAdd(p.wl.ready + run, 1);
      }
    }
  } else {
    // ===== epilogue (warps 4-11): warp -> TMEM lane quadrant q = warp % 4, column half hf
    const int q = warp & 3, hf = (warp - 4) >> 2;
    int acc_it = 0, p1_it = 0;
#ifdef CAEE_TILE_TRACE
    int cur = -1;
    for (;;) {
      if (cur >= 0 && cur < 4096 && threadIdx.x == 128) g_tile_trace[cur][5] = gtime();
      cur = tq.pop();
      if (!tm.at(cur, t)) break;
#else
    while (tm.at(tq.pop(), t)) {
#endif
      const int half_cols = ((p.wl.run_n[t.run] + 15) & ~15) >> 1;   // 8, 16, ..., 64
      if (half_cols <= 8) fp8_epilogue_tile<8>(p, t, tmem_base, tfull0, tempty0, acc_it, p1_it, amax_s, q, hf, lane, KS);
      else if (half_cols <= 16) fp8_epilogue_tile<16>(p, t, tmem_base, tfull0, tempty0, acc_it, p1_it, amax_s, q, hf, lane, KS);
      else if (half_cols <= 32) fp8_epilogue_tile<32>(p, t, tmem_base, tfull0, tempty0, acc_it, p1_it, amax_s, q, hf, lane, KS);
      else fp8_epilogue_tile<64>(p, t, tmem_base, tfull0, tempty0, acc_it, p1_it, amax_s, q, hf, lane, KS);
    }
  }

  tc_fence_before();
  __syncthreads();
  if (warp == 2) {
    tc_fence_after();
    asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;" ::"r"(tmem_base), "n"(kTmemCols));
  }
}

// ------------------------------------------------------------------ the kernel, part 2: epilogue of one tile
// The warp owns TMEM lanes [32 q, 32 q + 32) (weight rows of the tile) and token columns
// [hf CT, hf CT + CT).  Every 128-k block: wait for its accumulator pair, scale by
// w_scale[half, kb] * a_scale[token, kb], add into fp32 registers, hand the buffer back.
template <int CT>
__device__ __forceinline__ void fp8_epilogue_tile(const Fp8Params& p, const Tile& t, uint32_t tmem_base, uint32_t tfull0,
                                                  uint32_t tempty0, int& acc_it, int& p1_it, float (*amax_s)[kTileRows], int q,
                                                  int hf, int lane, int KS) {
  constexpr int NJ = CT > 32 ? 2 : 1;
  const int n = p.wl.run_n[t.run], start = p.wl.run_start[t.run], hrow = p.wl.run_hrow[t.run];
  const int nkb = t.phase == 1 ? p.KB1 / KS : p.KB2, kb0 = t.kq * nkb;      // kq = 0 unless a phase-1 tile's k range is split
  const int npad = (n + 15) & ~15;
  const int col0 = hf * CT, row = q * 32 + lane;
  const float* tab = reinterpret_cast<const float*>(p.packed[p.wl.run_expert[t.run]] + p.sc_off);
  const float* wsc = t.phase == 1 ? tab + ((size_t)t.sub * p.KB1 + kb0) * 2 : tab + p.t2_off + (size_t)t.sub * p.KB2 * 2;
  // activation scales: lane l fetches those of column col0 + l (+ 32), broadcast by shuffle below
  const float* abase[NJ];
#pragma unroll
  for (int j = 0; j < NJ; ++j) {
    const int cl = lane + 32 * j, col = col0 + cl;
    abase[j] = nullptr;
    if (cl < CT && col < n)
      abase[j] = t.phase == 1 ? p.xs + (size_t)p.wl.ent_tok[start + col] * p.KB1 + kb0 : p.hs + (size_t)(hrow + col) * p.KB2;
  }
  float acc0[CT], acc1[CT];
#pragma unroll
  for (int c = 0; c < CT; ++c) { acc0[c] = 0.f; acc1[c] = 0.f; }

  // h and its scales come from other SMs (L2 loads) and exist only once the run's phase-1 tiles
  // are done: the first completed accumulator proves it (the loaders waited for the run's
  // counter), so the scales of block kb + 1 are fetched while block kb is being added.
  float sv[NJ], sv_next[NJ];
#pragma unroll
  for (int j = 0; j < NJ; ++j) sv_next[j] = 0.f;
  for (int kb = 0; kb < nkb; ++kb, ++acc_it) {
    const int as = acc_it & 1;
    const float w0 = __ldg(wsc + kb * 2), w1 = __ldg(wsc + kb * 2 + 1);
    mbar_wait(tfull0 + 8 * as, (acc_it >> 1) & 1);
    tc_fence_after();
#pragma unroll
    for (int j = 0; j < NJ; ++j) {
      sv[j] = kb == 0 ? (abase[j] ? __ldcg(abase[j]) : 0.f) : sv_next[j];
      if (kb + 1 < nkb) sv_next[j] = abase[j] ? __ldcg(abase[j] + kb + 1) : 0.f;
    }
    const uint32_t taddr = tmem_base + ((uint32_t)(q * 32) << 16) + as * 256 + col0;
#pragma unroll
    for (int c0 = 0; c0 < CT; c0 += 8) {
      uint32_t d0[8], d1[8];
      tmem_ld8(taddr + c0, d0);
      tmem_ld8(taddr + 128 + c0, d1);
      if (CT <= 32) {   // hi and lo partial sums sit npad columns apart
        uint32_t e0[8], e1[8];
        tmem_ld8(taddr + npad + c0, e0);
        tmem_ld8(taddr + 128 + npad + c0, e1);
        tmem_ld_wait();
#pragma unroll
        for (int j = 0; j < 8; ++j) {
          d0[j] = __float_as_uint(__uint_as_float(d0[j]) + __uint_as_float(e0[j]));
          d1[j] = __float_as_uint(__uint_as_float(d1[j]) + __uint_as_float(e1[j]));
        }
      } else {
        tmem_ld_wait();
      }
#pragma unroll
      for (int j = 0; j < 8; ++j) {
        const int c = c0 + j;
        const float a = __shfl_sync(0xffffffffu, sv[c >> 5], c & 31);
        acc0[c] = fmaf(__uint_as_float(d0[j]), w0 * a, acc0[c]);
        acc1[c] = fmaf(__uint_as_float(d1[j]), w1 * a, acc1[c]);
      }
    }
    tc_fence_before();
    __syncwarp();
    if (lane == 0) mbar_arrive(tempty0 + 8 * as);
  }

  if (t.phase == 1 && KS > 1) {
    // split k range (KSplit, umma_common.cuh): leave this sub-tile's partial sums and count it; a reducer
    // warp finishes the tile (n <= kKSplitCols: CT == 8 and the hf == 0 warps hold every column)
    const int tile = (t.run - p.run_begin) * p.P1 + t.sub;
    CAEE_DEV_ASSERT(tile >= 0 && tile < p.ksp.tile_cap && n <= kKSplitCols);
    float* mine = p.ksp.part + ((size_t)tile * KS + t.kq) * (2 * kKSplitCols * kTileRows);
    if (hf == 0) {
#pragma unroll
      for (int c = 0; c < kKSplitCols; ++c) {
        if (c < n) {
          __stcg(mine + c * kTileRows + row, acc0[c]);
          __stcg(mine + (kKSplitCols + c) * kTileRows + row, acc1[c]);
        }
      }
    }
    asm volatile("bar.sync 3, 256;" ::: "memory");
    if (threadIdx.x == 128) {
      __threadfence();                        // cumulative: the CTA's partial stores, ordered by the barrier
      atomicAdd(p.ksp.cnt + tile, 1);
    }
    return;
  }
  if (t.phase == 1) {
    // h = silu(gate) * up; per-token maximum over the tile's 128 features -> the (token, k block)
    // scale of phase 2's activation operand; then the two e4m3 terms
    const int buf = p1_it % 3;
    unsigned* amax_u = reinterpret_cast<unsigned*>(amax_s[buf]);
#pragma unroll
    for (int c = 0; c < CT; ++c) {
      const float g = acc0[c], u = acc1[c];
      const float hv = col0 + c < n ? g / (1.0f + __expf(-g)) * u : 0.f;
      acc0[c] = hv;
      float m = fabsf(hv);
#pragma unroll
      for (int o = 16; o; o >>= 1) m = fmaxf(m, __shfl_xor_sync(0xffffffffu, m, o));
      if (lane == 0 && col0 + c < n) atomicMax(amax_u + col0 + c, __float_as_uint(m));
    }
    asm volatile("bar.sync 1, 256;" ::: "memory");
    if (lane < 16) amax_s[(p1_it + 2) % 3][(q + 4 * hf) * 16 + lane] = 0.f;   // the buffer of the tile after next
    uint8_t* hi_base = p.hq_hi + (size_t)hrow * p.I + t.sub * kTileRows + row;
    uint8_t* lo_base = p.hq_lo + (size_t)hrow * p.I + t.sub * kTileRows + row;
#pragma unroll
    for (int c = 0; c < CT; c += 2) {
      const int col = col0 + c;
      if (col < n) {
        const float m0 = amax_s[buf][col], m1 = col + 1 < n ? amax_s[buf][col + 1] : 0.f;
        const float s0 = m0 > 0.f ? m0 * (1.0f / 448.0f) : 1.0f, s1 = m1 > 0.f ? m1 * (1.0f / 448.0f) : 1.0f;
        const float v0 = acc0[c] / s0, v1 = acc0[c + 1] / s1;
        const uint16_t hi = cvt_e4m3x2(v0, v1);
        const float2 hf2 = e4m3x2_to_float2(hi);
        const uint16_t lo = cvt_e4m3x2(v0 - hf2.x, v1 - hf2.y);
        hi_base[(size_t)col * p.I] = (uint8_t)(hi & 0xff);
        lo_base[(size_t)col * p.I] = (uint8_t)(lo & 0xff);
        if (row == 0) p.hs[(size_t)(hrow + col) * p.KB2 + t.sub] = s0;
        if (col + 1 < n) {
          hi_base[(size_t)(col + 1) * p.I] = (uint8_t)(hi >> 8);
          lo_base[(size_t)(col + 1) * p.I] = (uint8_t)(lo >> 8);
          if (row == 0) p.hs[(size_t)(hrow + col + 1) * p.KB2 + t.sub] = s1;
        }
      }
    }
    ++p1_it;
    // publish this tile's slice of h: all 256 epilogue threads' stores (read later through the
    // async proxy by other SMs' TMA gathers), then one release add
    asm volatile("fence.proxy.async;" ::: "memory");
    __threadfence();
    asm volatile("bar.sync 2, 256;" ::: "memory");
    if (threadIdx.x == 128) atomicAdd(p.wl.ready + t.run, 1);
  } else {
    float* ocol = p.obuf + t.sub * 2 * kTileRows + row;
#pragma unroll
    for (int c = 0; c < CT; ++c) {
      const int col = col0 + c;
      if (col < n) {
        CAEE_DEV_ASSERT(p.wl.ent_dst[start + col] >= 0 && p.wl.ent_dst[start + col] < p.wl.ent_cap);
        float* o = caee_o_base(p.wl, p.obuf, p.wl.ent_tok[start + col]) + (ocol - p.obuf) + (size_t)p.wl.ent_dst[start + col] * p.H;
        o[0] = acc0[c];
        o[kTileRows] = acc1[c];
      }
    }
  }
}

#ifdef CAEE_TILE_TRACE
}  // namespace
extern "C" void caee_debug_tile_trace(long long* out, int n) { cudaMemcpyFromSymbol(out, g_tile_trace, sizeof(long long) * 6 * n); }
namespace {
#endif

size_t table_floats(const caee_ctx* c) {
  const int P1 = c->d.I / kTileRows, P2 = c->d.H / (2 * kTileRows), KS1 = c->d.H / kKBlock, KS2 = c->d.I / kKBlock;
  return (size_t)P1 * KS1 * 2 + (size_t)P2 * KS2 * 2;
}

}  // namespace

caee_status caee_fp8_supported(const caee_ctx* c, std::string* why) {
  const caee_layer_desc& d = c->d;
  if (d.H % 256 || d.I % 128) {
    *why = "the e4m3 UMMA expert kernel needs H % 256 == 0 and I % 128 == 0";
    return CAEE_ESHAPE;
  }
  return CAEE_OK;
}

size_t caee_fp8_packed_bytes(const caee_ctx* c) {
  return (size_t)3 * c->d.H * c->d.I + ((table_floats(c) * 4 + 15) & ~(size_t)15) + 16;   // + the 2^J pair
}

size_t caee_fp8_norm_offset(const caee_ctx* c) {
  return (size_t)3 * c->d.H * c->d.I + ((table_floats(c) * 4 + 15) & ~(size_t)15);
}

void caee_launch_pack_expert_fp8(caee_ctx* c, uint8_t* dst, const void* g, const void* u, const void* dn, const float* sg,
                                 const float* su, const float* sd, cudaStream_t st) {
  const int H = c->d.H, I = c->d.I;
  const size_t n1 = (size_t)I * (H / 16), n2 = (size_t)H * (I / 16);
  const size_t p2_off = (size_t)2 * I * H;
  k_pack_e4m3<<<(unsigned)((n1 + 255) / 256), 256, 0, st>>>((const uint8_t*)g, dst, I, H, 0, 0);
  k_pack_e4m3<<<(unsigned)((n1 + 255) / 256), 256, 0, st>>>((const uint8_t*)u, dst, I, H, 1, 0);
  k_pack_e4m3<<<(unsigned)((n2 + 255) / 256), 256, 0, st>>>((const uint8_t*)dn, dst, H, I, 2, p2_off);
  const int P1 = I / kTileRows, P2 = H / (2 * kTileRows);
  float* tab = reinterpret_cast<float*>(dst + (size_t)3 * H * I);
  k_scale_table<<<16, 256, 0, st>>>(sg, su, sd, tab, P1, P2, H / kKBlock, I / kKBlock);
  k_scale_norm<<<1, 256, 0, st>>>(tab, (int)table_floats(c), reinterpret_cast<float*>(dst + caee_fp8_norm_offset(c)));
}

// 2D byte tensor maps over the [hi rows | lo rows] x k arrays of x and h for tile::gather4 row
// gathers: box = one row of 128 bytes, 128-byte swizzle (the layout the MMA descriptor names).
caee_status caee_fp8_make_tensor_maps(caee_ctx* c) {
  if (!encode_row_gather_map(c->tm_x, c->xq, (size_t)c->d.H, (size_t)2 * c->d.max_tokens) ||
      !encode_row_gather_map(c->tm_h, c->hq, (size_t)c->d.I, (size_t)2 * c->h_rows_cap))
    return caee_fail(c, CAEE_ECUDA, "cuTensorMapEncodeTiled failed for the e4m3 token-operand maps");
  c->tm_ready = true;
  return CAEE_OK;
}

// Once per step, before the first expert launch: x -> its two e4m3 terms and block scales.
void caee_launch_fp8_prepare(caee_ctx* c, const void* x, int T, cudaStream_t st) {
  if (T <= 0) return;
  ++c->n_launches;
  const size_t n_blocks = (size_t)T * (c->d.H / kKBlock);
  const size_t TH = (size_t)c->d.max_tokens * c->d.H;
  k_act_split<<<(unsigned)((n_blocks + 7) / 8), 256, 0, st>>>((const __nv_bfloat16*)x, c->xq, c->xq + TH, c->xs, n_blocks);
}

// runs [run_begin, run_begin + run_count) (run_count < 0: every run of the work list), tile
// tickets from wl.sched[ticket].
void caee_launch_expert_fp8(caee_ctx* c, int T, int run_begin, int run_count, int ticket, cudaStream_t st) {
  const caee_layer_desc& d = c->d;
  Fp8Params p;
  p.wl = c->wl;
  p.packed = c->packed.dev_ptrs;
  const size_t TH = (size_t)d.max_tokens * d.H, RI = c->h_rows_cap * (size_t)d.I;
  p.xq_hi = c->xq; p.xq_lo = c->xq + TH; p.xs = c->xs;
  p.hq_hi = c->hq; p.hq_lo = c->hq + RI; p.hs = c->hs;
  p.obuf = c->obuf;
  p.H = d.H; p.I = d.I;
  p.P1 = d.I / kTileRows; p.P2 = d.H / (2 * kTileRows);
  p.KB1 = d.H / kKBlock; p.KB2 = d.I / kKBlock;
  p.run_begin = run_begin; p.run_count = run_count; p.ticket = ticket;
  p.sc_off = (int)((size_t)3 * d.H * d.I);
  p.t2_off = p.P1 * p.KB1 * 2;
  memcpy(&p.tm_x, c->tm_x, sizeof(CUtensorMap));
  memcpy(&p.tm_h, c->tm_h, sizeof(CUtensorMap));
  p.lo_row_x = d.max_tokens;
  p.lo_row_h = (int)c->h_rows_cap;
  const int ncap = std::min((int)c->wl.run_cap, (T + 15) & ~15);
  p.b_term_bytes = ncap * kKBlock;                  // one e4m3 term of the token operand
  p.stage_bytes = kAStageBytes + 2 * p.b_term_bytes;
  const int max_dyn = 227 * 1024 - 4096;            // leave room for the static barriers / amax buffers
  p.n_stages = std::min(kMaxStages, (max_dyn - 1024) / p.stage_bytes);
  const size_t dyn = (size_t)p.n_stages * p.stage_bytes + 1024;
  p.ksp = caee_ksplit_for(c, T, p.KB1, ticket);
  if (!(c->attr_done & 2u)) {
    cudaFuncSetAttribute(k_expert_fp8, cudaFuncAttributeMaxDynamicSharedMemorySize, max_dyn);
    c->attr_done |= 2u;
  }
  ++c->n_launches;
  if (c->pdl && !c->any_offload) {
    // programmatic dependent launch behind the decision kernel (the x split runs before the router GEMM)
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = dim3((unsigned)c->num_sms);
    cfg.blockDim = dim3(kThreads);
    cfg.dynamicSmemBytes = dyn;
    cfg.stream = st;
    cudaLaunchAttribute at[1];
    at[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    at[0].val.programmaticStreamSerializationAllowed = 1;
    cfg.attrs = at; cfg.numAttrs = 1;
    cudaLaunchKernelEx(&cfg, k_expert_fp8, p);
    return;
  }
  k_expert_fp8<<<c->num_sms, kThreads, dyn, st>>>(p);
}
