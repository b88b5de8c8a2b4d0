// expert_umma.cu — S7 grouped SwiGLU expert FFN for sm_100a: a persistent, warp-specialised
// kernel that streams each surviving expert's weights from HBM exactly once with the bulk
// async-copy engine (TMA, cp.async.bulk -> SASS UBLKCP) into a multi-stage shared-memory ring
// and contracts them on the 5th-gen tensor cores (tcgen05.mma, accumulators in TMEM).
//
// Why this shape.  At decode (1-128 tokens) an expert sees a handful of tokens, so the work
// is one pass over 3*H*I weight elements per surviving expert and the bound is HBM bandwidth
// (Fig. 1).  The contraction is put on the tensor cores "swapped": the
// 128 weight rows of a tile are the MMA M dimension, the (padded) tokens are N (16..128), so a
// tiny batch still fills an instruction and the tensor pipe stays far below its limit.
// Pruned experts never appear in the work list, so their bytes are never requested.
//
// Layout.  caee_set_weights(pack=1) rewrites every expert once into "stage images": each
// 32 KB stage is two 128-row x 64-k bf16 tiles in the UMMA canonical K-major, no-swizzle
// core-matrix order (8 rows x 16 B contiguous = one 128 B core matrix; LBO = 128 B between
// k-adjacent core matrices, SBO = 1024 B between 8-row groups).  A stage is therefore ONE
// contiguous 32 KB bulk copy, and consecutive stages of a tile are consecutive in HBM.
//   phase 1 (gate/up):  tile ft = features [128 ft, 128 ft + 128), stage kb = k in [64 kb, +64):
//                       [gate tile][up tile]      -> D0 = gate rows, D1 = up rows (TMEM)
//   phase 2 (down):     tile op = out rows [256 op, +256), stage kb over I:
//                       [rows +0..127][rows +128..255] -> D0, D1
// B operand (tokens): x rows (phase 1) or h rows (phase 2), gathered by two loader warps with
// ordinary loads (they are L2-resident and 0.1% of the bytes) into the same canonical layout.
//
// FP8 (e4m3 weights, 128x128 block scales, BASELINE.json config 4).  The HBM stream is the raw
// e4m3 bytes: a stage image is 16 KB (two 128-row x 64-k tiles, 8-row x 16-byte core blocks) and
// lands in a separate "landing" ring.  Four converter warps widen each landing stage to fp16
// (cvt.rn.f16x2.e4m3x2 is exact) times ratio = scale[tile, k-block] / ref[tile] (ref = the
// tile's largest block scale, so ratio <= 1 and nothing leaves the fp16 range; one fp16 rounding,
// 2^-11) into the same canonical 32 KB operand stage the bf16 path uses; the tensor cores then
// run kind::f16 on fp16 weights x fp16 activations (x is widened bf16->fp16 once per step, h is
// written as fp16) with fp32 accumulation, and the epilogue multiplies each accumulator row by
// its tile's ref.  Quantising the activations to e4m3 instead would not meet the 5e-2 x RMS
// tolerance, and HBM traffic is what counts at decode: 1 byte per weight.
//
// Roles (256 threads, +128 converter threads for FP8; 1 CTA per SM):  warp 0 = weight producer (one lane issues bulk copies),
// warp 1 = MMA issuer (one lane), warps 2-3 = token-operand loaders (warp 2 also owns TMEM
// alloc/free), warps 4-7 = epilogue (TMEM -> registers -> SwiGLU -> h, or -> o rows).
// Tiles are claimed dynamically (one atomic ticket per tile, phase-1 tickets first); a
// phase-2 tile only waits (per-run counter) for phase-1 tiles, which never wait, so the
// schedule cannot deadlock and CTAs that finish early simply claim more tiles.
#include "caee_internal.cuh"

namespace {

constexpr int kThreads = 256;
constexpr int kThreadsFp8 = 384;        // + 4 converter warps
constexpr int kLandBytes = 16 * 1024;   // one e4m3 stage image (two 128 x 64 tiles)
constexpr int kMaxRatio = 256;          // floats of block-scale ratios per tile (2 per 128-k block)
constexpr int kTileRows = 128;          // UMMA M
constexpr int kKBlock = 64;             // k elements per stage
constexpr int kATileBytes = kTileRows * kKBlock * 2;  // 16 KB
constexpr int kAStageBytes = 2 * kATileBytes;         // 32 KB: two tiles per stage
constexpr int kTmemCols = 512;
constexpr int kMaxStages = 8;

struct UmmaParams {
  caee_worklist wl;
  uint8_t* const* packed;     // [E+S] stage images
  const uint16_t* x;          // [T,H] bf16 (bf16 weights) or its fp16 copy (e4m3 weights)
  uint16_t* hbuf;             // [rows,I] bf16 / fp16
  float* obuf;                // [T*(k+S),H]
  int H, I;
  int P1, P2, KB1, KB2;       // tiles per run and 64-k stages per tile, per phase
  int n_stages, b_stage_bytes, stage_bytes;
  int n_land, land_off;       // FP8: landing ring (stages, byte offset in dynamic smem)
  int run_begin, run_count;   // runs [run_begin, run_begin + run_count) of the work list; run_count < 0: all
  int ticket;                 // which tile-ticket counter of wl.sched this launch uses
  int sc_off, r2_off;         // FP8: byte offset of the scale tables in a packed image; float offset of the phase-2 part
};

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
__device__ __forceinline__ uint4 lds128(uint32_t a) {
  uint4 v;
  asm volatile("ld.shared.v4.u32 {%0,%1,%2,%3}, [%4];" : "=r"(v.x), "=r"(v.y), "=r"(v.z), "=r"(v.w) : "r"(a));
  return v;
}
__device__ __forceinline__ void sts128(uint32_t a, uint32_t x, uint32_t y, uint32_t z, uint32_t w) {
  asm volatile("st.shared.v4.u32 [%0], {%1,%2,%3,%4};" ::"r"(a), "r"(x), "r"(y), "r"(z), "r"(w) : "memory");
}
// four e4m3 codes (k ascending from the low byte) -> four fp16 values times r, as two packed words
__device__ __forceinline__ void widen_e4m3x4(uint32_t w, __half2 r, uint32_t& o0, uint32_t& o1) {
  uint32_t a, b;
  asm("cvt.rn.f16x2.e4m3x2 %0, %1;" : "=r"(a) : "h"((uint16_t)(w & 0xffffu)));
  asm("cvt.rn.f16x2.e4m3x2 %0, %1;" : "=r"(b) : "h"((uint16_t)(w >> 16)));
  __half2 ha = __hmul2(*reinterpret_cast<__half2*>(&a), r), hb = __hmul2(*reinterpret_cast<__half2*>(&b), r);
  o0 = *reinterpret_cast<uint32_t*>(&ha);
  o1 = *reinterpret_cast<uint32_t*>(&hb);
}

__device__ __forceinline__ int ld_acquire(const int* p) {
  int v;
  asm volatile("ld.acquire.gpu.global.s32 %0, [%1];" : "=r"(v) : "l"(p) : "memory");
  return v;
}
struct Tile {
  int phase, run, sub;  // sub = ft (phase 1) or op (phase 2)
};
struct TileMap {
  int n_runs, run_begin, P1, P2;
  __device__ __forceinline__ bool at(int i, Tile& t) const {
    const int t1 = n_runs * P1;
    if (i < t1) { const int r = i / P1; t.phase = 1; t.sub = i - r * P1; t.run = run_begin + r; return true; }
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
};

template <bool kFp8>
__global__ void __launch_bounds__(kFp8 ? kThreadsFp8 : kThreads, 1) k_expert_umma(const UmmaParams p) {
  extern __shared__ __align__(1024) uint8_t smem_raw[];
  uint8_t* smem = reinterpret_cast<uint8_t*>((reinterpret_cast<uintptr_t>(smem_raw) + 1023) & ~(uintptr_t)1023);
  __shared__ __align__(8) uint64_t bars[4 * kMaxStages + 4 + 2 * kQueue];
  __shared__ uint32_t tmem_base_s;
  __shared__ int tq_slots[kQueue];
  __shared__ float ratio_s[kFp8 ? 2 * kMaxRatio : 1];

  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const uint32_t smem_base = smem_u32(smem);
  const uint32_t full0 = smem_u32(&bars[0]), empty0 = smem_u32(&bars[kMaxStages]);
  const uint32_t tfull0 = smem_u32(&bars[2 * kMaxStages]), tempty0 = smem_u32(&bars[2 * kMaxStages + 2]);
  const uint32_t qfull0 = smem_u32(&bars[2 * kMaxStages + 4]), qempty0 = smem_u32(&bars[2 * kMaxStages + 4 + kQueue]);
  const uint32_t lfull0 = smem_u32(&bars[2 * kMaxStages + 4 + 2 * kQueue]), lempty0 = lfull0 + 8 * kMaxStages;
  const TileMap tm{p.run_count >= 0 ? p.run_count : p.wl.meta[1], p.run_begin, p.P1, p.P2};

  if (threadIdx.x == 0) {
    for (int s = 0; s < p.n_stages; ++s) {
      // bf16: producer's expect_tx arrive + 2 loader warps; fp8: 4 converter warps + 2 loader warps
      mbar_init(full0 + 8 * s, kFp8 ? 6 : 3);
      mbar_init(empty0 + 8 * s, 1);  // tcgen05.commit
    }
    if (kFp8)
      for (int s = 0; s < p.n_land; ++s) {
        mbar_init(lfull0 + 8 * s, 1);   // producer's expect_tx arrive
        mbar_init(lempty0 + 8 * s, 4);  // converter warps
      }
    for (int a = 0; a < 2; ++a) {
      mbar_init(tfull0 + 8 * a, 1);   // tcgen05.commit
      mbar_init(tempty0 + 8 * a, 4);  // one lane of each epilogue warp
    }
    for (int q = 0; q < kQueue; ++q) {
      mbar_init(qfull0 + 8 * q, 1);                // producer
      mbar_init(qempty0 + 8 * q, kFp8 ? 11 : 7);   // MMA warp + 2 loader warps + 4 epilogue warps (+ 4 converters)
    }
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
  }
  if (warp == 2) {
    asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], %1;" ::"r"(smem_u32(&tmem_base_s)),
                 "n"(kTmemCols));
    asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;");
  }
  tc_fence_before();
  __syncthreads();
  tc_fence_after();
  const uint32_t tmem_base = tmem_base_s;
  TileQueue tq{qfull0, qempty0, tq_slots, 0, 0};
  Tile t;
  constexpr int kSrcStage = kFp8 ? kLandBytes : kAStageBytes;  // bytes of one stage image in HBM

  if (warp == 0) {
    // ===== weight producer: claims tiles; one bulk copy per stage from the packed image
    if (lane == 0) {
      int stage = 0, ph = 0, q = 0, qph = 0;
      const int ring = kFp8 ? p.n_land : p.n_stages;
      for (;;) {
        mbar_wait(qempty0 + 8 * q, qph ^ 1);
        const int i = atomicAdd(p.wl.sched + p.ticket, 1);
        tq_slots[q] = i;
        mbar_arrive(qfull0 + 8 * q);
        if (++q == kQueue) { q = 0; qph ^= 1; }
        if (!tm.at(i, t)) break;
        const int e = p.wl.run_expert[t.run];
        const int nkb = t.phase == 1 ? p.KB1 : p.KB2;
        const uint8_t* src = p.packed[e] + (t.phase == 1 ? (size_t)t.sub * p.KB1 : (size_t)p.P1 * p.KB1 + (size_t)t.sub * p.KB2) * kSrcStage;
        for (int kb = 0; kb < nkb; ++kb) {
          if (kFp8) {
            mbar_wait(lempty0 + 8 * stage, ph ^ 1);
            mbar_arrive_expect_tx(lfull0 + 8 * stage, kLandBytes);
            bulk_g2s(smem_base + p.land_off + stage * kLandBytes, src + (size_t)kb * kLandBytes, kLandBytes, lfull0 + 8 * stage);
          } else {
            mbar_wait(empty0 + 8 * stage, ph ^ 1);
            mbar_arrive_expect_tx(full0 + 8 * stage, kAStageBytes);
            bulk_g2s(smem_base + stage * p.stage_bytes, src + (size_t)kb * kAStageBytes, kAStageBytes, full0 + 8 * stage);
          }
          if (++stage == ring) { stage = 0; ph ^= 1; }
        }
      }
    }
  } else if (warp == 1) {
    // ===== MMA issuer (the whole warp pops the queue; one lane issues)
    int stage = 0, ph = 0;
    for (int it = 0; tm.at(tq.pop(), t); ++it) {
      if (lane == 0) {
        const int as = it & 1;
        const int npad = (p.wl.run_n[t.run] + 15) & ~15;
        const uint32_t idesc = make_idesc(npad, !kFp8);
        const int nkb = t.phase == 1 ? p.KB1 : p.KB2;
        mbar_wait(tempty0 + 8 * as, ((it >> 1) & 1) ^ 1);
        tc_fence_after();
        const uint32_t d0 = tmem_base + as * 256, d1 = d0 + 128;
        for (int kb = 0; kb < nkb; ++kb) {
          mbar_wait(full0 + 8 * stage, ph);
          tc_fence_after();
          const uint32_t a_addr = smem_base + stage * p.stage_bytes;
          const uint64_t a0 = make_desc(a_addr), a1 = make_desc(a_addr + kATileBytes), b = make_desc(a_addr + kAStageBytes);
#pragma unroll
          for (int ks = 0; ks < kKBlock / 16; ++ks) {
            const uint32_t acc = (kb | ks) ? 1u : 0u;
            umma_bf16(d0, a0 + (uint64_t)(ks * 16), b + (uint64_t)(ks * 16), idesc, acc);  // +256 B per k-step (>>4)
            umma_bf16(d1, a1 + (uint64_t)(ks * 16), b + (uint64_t)(ks * 16), idesc, acc);
          }
          tc_commit(empty0 + 8 * stage);
          if (++stage == p.n_stages) { stage = 0; ph ^= 1; }
        }
        tc_commit(tfull0 + 8 * as);
      } else {
        // keep the ring position in step with lane 0
        const int nkb = t.phase == 1 ? p.KB1 : p.KB2;
        stage = (stage + nkb) % p.n_stages;
      }
      __syncwarp();
    }
  } else if (warp == 2 || warp == 3) {
    // ===== token-operand loaders: gather B rows (x or h) into the canonical K-major layout with
    // cp.async, kLag stages in flight per warp so that L2 latency is off the critical path
    const int wq = warp - 2;
    const int r8 = lane & 7, c4 = lane >> 3;  // row in 8-row group, 16-byte chunk (c4 and c4+4)
    int stage = 0, ph = 0, pend_stage = 0, pending = 0;
    const int lag = min(kLag, p.n_stages - 1);  // a stage is published `lag` stages late: must stay inside the ring
    auto publish = [&](int count) {  // the oldest `count` in-flight stages have landed
      fence_proxy_async_smem();
      __syncwarp();
      for (int j = 0; j < count; ++j) {
        if (lane == 0) mbar_arrive(full0 + 8 * pend_stage);
        if (++pend_stage == p.n_stages) pend_stage = 0;
      }
      pending -= count;
    };
    while (tm.at(tq.pop(), t)) {
      const int n = p.wl.run_n[t.run], start = p.wl.run_start[t.run];
      const int ngroups = (n + 15) / 16 * 2;  // 8-row groups in the padded tile
      const int nkb = t.phase == 1 ? p.KB1 : p.KB2;
      const uint8_t* rowp[8];  // this lane's source row in each of its groups (nullptr: zero fill)
#pragma unroll
      for (int g = 0; g < 8; ++g) {
        const int row = (2 * g + wq) * 8 + r8;
        rowp[g] = nullptr;
        if (row < n) {
          if (t.phase == 1) rowp[g] = reinterpret_cast<const uint8_t*>(p.x + (size_t)p.wl.ent_tok[start + row] * p.H);
          else rowp[g] = reinterpret_cast<const uint8_t*>(p.hbuf + (size_t)(p.wl.run_hrow[t.run] + row) * p.I);
        }
      }
      if (t.phase == 2) {
        // h of this run is complete once all P1 gate/up tiles have published it
        if (lane == 0) {
          const int* flag = p.wl.ready + t.run;
          while (ld_acquire(flag) < p.P1) __nanosleep(64);
        }
        __syncwarp();
      }
      for (int kb = 0; kb < nkb; ++kb) {
        mbar_wait(empty0 + 8 * stage, ph ^ 1);
        const uint32_t b_addr = smem_base + stage * p.stage_bytes + kAStageBytes;
#pragma unroll
        for (int g = 0; g < 8; ++g) {
          if (2 * g + wq < ngroups) {
            const uint32_t a = b_addr + (2 * g + wq) * 1024 + r8 * 16;
            const uint8_t* src = rowp[g] ? rowp[g] + (size_t)kb * 128 + c4 * 16 : reinterpret_cast<const uint8_t*>(p.x);
            const uint32_t sz = rowp[g] ? 16u : 0u;  // src-size 0: zero fill
            asm volatile("cp.async.cg.shared.global [%0], [%1], 16, %2;" ::"r"(a + c4 * 128), "l"(src), "r"(sz) : "memory");
            asm volatile("cp.async.cg.shared.global [%0], [%1], 16, %2;" ::"r"(a + (c4 + 4) * 128), "l"(src + (rowp[g] ? 64 : 0)), "r"(sz) : "memory");
          }
        }
        asm volatile("cp.async.commit_group;" ::: "memory");
        ++pending;
        if (++stage == p.n_stages) { stage = 0; ph ^= 1; }
        if (pending > lag) {
          if (lag >= 3) asm volatile("cp.async.wait_group 3;" ::: "memory");
          else if (lag == 2) asm volatile("cp.async.wait_group 2;" ::: "memory");
          else asm volatile("cp.async.wait_group 1;" ::: "memory");
          publish(1);
        }
      }
      // flush at the tile boundary: nothing of this tile may wait behind a later tile's dependency
      asm volatile("cp.async.wait_group 0;" ::: "memory");
      publish(pending);
    }
  } else if (warp < 8) {
    // ===== epilogue: TMEM -> registers -> SwiGLU -> h (phase 1) or -> o rows (phase 2)
    const int q = warp - 4;  // TMEM lane quadrant of this warp (warp % 4)
    for (int it = 0; tm.at(tq.pop(), t); ++it) {
      const int as = it & 1;
      const int n = p.wl.run_n[t.run], start = p.wl.run_start[t.run];
      float ref0 = 1.f, ref1 = 1.f;  // FP8: the tile's reference block scales (rows of D0 / D1)
      if (kFp8) {
        const float* tab = reinterpret_cast<const float*>(p.packed[p.wl.run_expert[t.run]] + p.sc_off);
        const float* rp = t.phase == 1 ? tab + (size_t)p.P1 * (p.H / 128) * 2 + t.sub * 2
                                       : tab + p.r2_off + (size_t)p.P2 * (p.I / 128) * 2 + t.sub * 2;
        ref0 = rp[0];
        ref1 = rp[1];
      }
      mbar_wait(tfull0 + 8 * as, (it >> 1) & 1);
      tc_fence_after();
      const uint32_t tbase = tmem_base + ((uint32_t)(q * 32) << 16) + as * 256;
      const int row = q * 32 + lane;
      if (t.phase == 1) {
        uint16_t* hcol = p.hbuf + (size_t)p.wl.run_hrow[t.run] * p.I + t.sub * kTileRows + row;
        for (int c = 0; c < n; c += 16) {
          uint32_t g[16], u[16];
          tmem_ld16(tbase + c, g);
          tmem_ld16(tbase + 128 + c, u);
          tmem_ld_wait();
#pragma unroll
          for (int j = 0; j < 16; ++j) {
            if (c + j < n) {
              const float gv = __uint_as_float(g[j]) * ref0, uv = __uint_as_float(u[j]) * ref1;
              const float hv = gv / (1.0f + __expf(-gv)) * uv;
              hcol[(size_t)(c + j) * p.I] = kFp8 ? __half_as_ushort(__float2half_rn(hv))
                                                 : __bfloat16_as_ushort(__float2bfloat16_rn(hv));
            }
          }
        }
      } else {
        float* ocol = p.obuf + t.sub * 2 * kTileRows + row;
        for (int c = 0; c < n; c += 16) {
          uint32_t d0[16], d1[16];
          tmem_ld16(tbase + c, d0);
          tmem_ld16(tbase + 128 + c, d1);
          tmem_ld_wait();
#pragma unroll
          for (int j = 0; j < 16; ++j) {
            if (c + j < n) {
              float* o = ocol + (size_t)p.wl.ent_dst[start + c + j] * p.H;
              o[0] = __uint_as_float(d0[j]) * ref0;
              o[kTileRows] = __uint_as_float(d1[j]) * ref1;
            }
          }
        }
      }
      tc_fence_before();
      __syncwarp();
      if (lane == 0) mbar_arrive(tempty0 + 8 * as);
      if (t.phase == 1) {
        // publish this tile's slice of h: all 128 epilogue threads' stores, then one release add
        __threadfence();
        asm volatile("bar.sync 1, 128;" ::: "memory");
        if (threadIdx.x == 128) atomicAdd(p.wl.ready + t.run, 1);
      }
    }
  } else if (kFp8) {
    // ===== converters (FP8 only): landing stage (e4m3) -> operand stage (fp16 x block-scale ratio)
    const int cw = warp - 8;
    int cs = 0, cph = 0, ls = 0, lph = 0;
    for (int it = 0; tm.at(tq.pop(), t); ++it) {
      const int nkb = t.phase == 1 ? p.KB1 : p.KB2;
      const int nr = (t.phase == 1 ? p.H : p.I) / 128 * 2;  // (ratio D0, ratio D1) per 128-k block
      const float* tab = reinterpret_cast<const float*>(p.packed[p.wl.run_expert[t.run]] + p.sc_off);
      const float* rr = t.phase == 1 ? tab + (size_t)t.sub * nr : tab + p.r2_off + (size_t)t.sub * nr;
      float* rs = ratio_s + (it & 1) * kMaxRatio;
      for (int i = threadIdx.x - 256; i < nr; i += 128) rs[i] = rr[i];
      asm volatile("bar.sync 2, 128;" ::: "memory");
      for (int kb = 0; kb < nkb; ++kb) {
        mbar_wait(lfull0 + 8 * ls, lph);
        mbar_wait(empty0 + 8 * cs, cph ^ 1);
        const __half2 r0 = __float2half2_rn(rs[(kb >> 1) * 2]), r1 = __float2half2_rn(rs[(kb >> 1) * 2 + 1]);
        const uint32_t land = smem_base + p.land_off + ls * kLandBytes + lane * 16;
        const uint32_t conv = smem_base + cs * p.stage_bytes + (lane >> 3) * 256 + (lane & 7) * 16;
#pragma unroll
        for (int j = 0; j < 8; ++j) {
          const int g = cw * 8 + j;  // 8-row group 0..31: 0-15 first tile, 16-31 second tile
          const uint4 v = lds128(land + g * 512);
          const __half2 r = g < 16 ? r0 : r1;
          uint32_t o[8];
          widen_e4m3x4(v.x, r, o[0], o[1]);
          widen_e4m3x4(v.y, r, o[2], o[3]);
          widen_e4m3x4(v.z, r, o[4], o[5]);
          widen_e4m3x4(v.w, r, o[6], o[7]);
          const uint32_t dst = conv + (g >> 4) * kATileBytes + (g & 15) * 1024;
          sts128(dst, o[0], o[1], o[2], o[3]);
          sts128(dst + 128, o[4], o[5], o[6], o[7]);
        }
        fence_proxy_async_smem();
        __syncwarp();
        if (lane == 0) {
          mbar_arrive(full0 + 8 * cs);
          mbar_arrive(lempty0 + 8 * ls);
        }
        if (++cs == p.n_stages) { cs = 0; cph ^= 1; }
        if (++ls == p.n_land) { ls = 0; lph ^= 1; }
      }
    }
  }

  tc_fence_before();
  __syncthreads();
  if (warp == 2) {
    tc_fence_after();
    asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;" ::"r"(tmem_base), "n"(kTmemCols));
  }
}

// One thread per 16-byte chunk: raw row-major [rows, cols] bf16 -> stage images.
// which: 0 gate, 1 up (phase-1 region), 2 down (phase-2 region).
__global__ void __launch_bounds__(256) k_pack_bf16(const __nv_bfloat16* __restrict__ src, uint8_t* __restrict__ dst, int rows,
                                                   int cols, int which, size_t region_off) {
  const size_t chunk = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
  const int cpr = cols / 8;
  if (chunk >= (size_t)rows * cpr) return;
  const int r = (int)(chunk / cpr), k0 = (int)(chunk % cpr) * 8;
  const int kb = k0 / kKBlock, kk = k0 % kKBlock, nkb = cols / kKBlock;
  size_t stage, in_stage;
  if (which < 2) {
    const int ft = r / kTileRows, rr = r % kTileRows;
    stage = (size_t)ft * nkb + kb;
    in_stage = (size_t)which * kATileBytes + (rr / 8) * 1024 + (kk / 8) * 128 + (rr % 8) * 16;
  } else {
    const int op = r / (2 * kTileRows), half = (r / kTileRows) & 1, rr = r % kTileRows;
    stage = (size_t)op * nkb + kb;
    in_stage = (size_t)half * kATileBytes + (rr / 8) * 1024 + (kk / 8) * 128 + (rr % 8) * 16;
  }
  const uint4 v = *reinterpret_cast<const uint4*>(src + (size_t)r * cols + k0);
  *reinterpret_cast<uint4*>(dst + region_off + stage * kAStageBytes + in_stage) = v;
}

// Same for e4m3: one thread per 16 codes; a stage image is 16 KB = two 8 KB tiles of
// 8-row x 16-byte core blocks ([8-row group][16-k chunk][row][16 B]).
__global__ void __launch_bounds__(256) k_pack_e4m3(const uint8_t* __restrict__ src, uint8_t* __restrict__ dst, int rows,
                                                   int cols, int which, size_t region_off) {
  const size_t chunk = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
  const int cpr = cols / 16;
  if (chunk >= (size_t)rows * cpr) return;
  const int r = (int)(chunk / cpr), k0 = (int)(chunk % cpr) * 16;
  const int kb = k0 / kKBlock, kk = k0 % kKBlock, nkb = cols / kKBlock;
  int tile, half, rr = r % kTileRows;
  if (which < 2) { tile = r / kTileRows; half = which; }
  else { tile = r / (2 * kTileRows); half = (r / kTileRows) & 1; }
  const size_t stage = (size_t)tile * nkb + kb;
  const size_t in_stage = (size_t)half * (kLandBytes / 2) + (rr / 8) * 512 + (kk / 16) * 128 + (rr % 8) * 16;
  const uint4 v = *reinterpret_cast<const uint4*>(src + (size_t)r * cols + k0);
  *reinterpret_cast<uint4*>(dst + region_off + stage * kLandBytes + in_stage) = v;
}

// Block-scale tables of one expert (see UmmaParams::sc_off): for each tile the per-128-k-block
// ratio scale/ref of its two 128-row halves, and ref = the half's largest block scale.
//   phase 1, tile ft:  halves = gate rows / up rows of feature block ft   (scale row ft of each)
//   phase 2, tile op:  halves = down rows 256 op + [0,128) / + [128,256)  (scale rows 2 op, 2 op + 1)
__global__ void k_scale_tables(const float* __restrict__ sg, const float* __restrict__ su, const float* __restrict__ sd,
                               float* __restrict__ tab, int P1, int P2, int KS1, int KS2) {
  const int tile = blockIdx.x, half = threadIdx.x;  // 2 threads per block
  const bool ph1 = tile < P1;
  const int t = ph1 ? tile : tile - P1, KS = ph1 ? KS1 : KS2;
  const float* row = ph1 ? (half == 0 ? sg : su) + (size_t)t * KS1 : sd + (size_t)(2 * t + half) * KS2;
  float* ratio = tab + (ph1 ? (size_t)t * KS1 * 2 : (size_t)P1 * KS1 * 2 + P1 * 2 + (size_t)t * KS2 * 2);
  float* ref = tab + (ph1 ? (size_t)P1 * KS1 * 2 + t * 2 : (size_t)P1 * KS1 * 2 + P1 * 2 + (size_t)P2 * KS2 * 2 + t * 2);
  float m = 0.f;
  for (int j = 0; j < KS; ++j) m = fmaxf(m, fabsf(row[j]));
  for (int j = 0; j < KS; ++j) ratio[j * 2 + half] = m > 0.f ? row[j] / m : 0.f;
  ref[half] = m;
}

__global__ void __launch_bounds__(256) k_bf16_to_f16(const __nv_bfloat16* __restrict__ x, __half* __restrict__ out, size_t n) {
  const size_t i = ((size_t)blockIdx.x * blockDim.x + threadIdx.x) * 2;
  if (i + 1 < n) {
    const __nv_bfloat162 v = *reinterpret_cast<const __nv_bfloat162*>(x + i);
    *reinterpret_cast<__half2*>(out + i) = __floats2half2_rn(__low2float(v), __high2float(v));
  } else if (i < n) {
    out[i] = __float2half_rn(__bfloat162float(x[i]));
  }
}

size_t table_floats(const caee_ctx* c) {
  const int P1 = c->d.I / kTileRows, P2 = c->d.H / (2 * kTileRows), KS1 = c->d.H / 128, KS2 = c->d.I / 128;
  return (size_t)P1 * KS1 * 2 + P1 * 2 + (size_t)P2 * KS2 * 2 + P2 * 2;
}

}  // namespace

caee_status caee_umma_supported(const caee_ctx* c, std::string* why) {
  const caee_layer_desc& d = c->d;
  if ((d.w_dtype != CAEE_BF16 && d.w_dtype != CAEE_E4M3) || d.act_dtype != CAEE_BF16) {
    *why = "the UMMA expert kernel takes bf16 or e4m3 weights and bf16 activations";
    return CAEE_EDTYPE;
  }
  if (d.H % 256 || d.I % 128) {
    *why = "the UMMA expert kernel needs H % 256 == 0 and I % 128 == 0";
    return CAEE_ESHAPE;
  }
  if (d.w_dtype == CAEE_E4M3) return caee_fp8_supported(c, why);
  return CAEE_OK;
}

size_t caee_umma_packed_bytes(const caee_ctx* c) {
  const size_t elems = (size_t)3 * c->d.H * c->d.I;
  if (c->d.w_dtype == CAEE_BF16) return elems * 2;
  return caee_fp8_packed_bytes(c);
}

void caee_launch_pack_expert(caee_ctx* c, int e, uint8_t* dst, const void* g, const void* u, const void* dn, const float* sg,
                             const float* su, const float* sd, cudaStream_t st) {
  (void)e;
  const int H = c->d.H, I = c->d.I;
  if (c->d.w_dtype == CAEE_E4M3) {
    caee_launch_pack_expert_fp8(c, dst, g, u, dn, sg, su, sd, st);
    return;
  }
  if (c->d.w_dtype == CAEE_BF16) {
    const size_t n1 = (size_t)I * (H / 8), n2 = (size_t)H * (I / 8);
    const size_t p2_off = (size_t)2 * I * H * 2;
    k_pack_bf16<<<(unsigned)((n1 + 255) / 256), 256, 0, st>>>((const __nv_bfloat16*)g, dst, I, H, 0, 0);
    k_pack_bf16<<<(unsigned)((n1 + 255) / 256), 256, 0, st>>>((const __nv_bfloat16*)u, dst, I, H, 1, 0);
    k_pack_bf16<<<(unsigned)((n2 + 255) / 256), 256, 0, st>>>((const __nv_bfloat16*)dn, dst, H, I, 2, p2_off);
  } else {
    const size_t n1 = (size_t)I * (H / 16), n2 = (size_t)H * (I / 16);
    const size_t p2_off = (size_t)2 * I * H;
    k_pack_e4m3<<<(unsigned)((n1 + 255) / 256), 256, 0, st>>>((const uint8_t*)g, dst, I, H, 0, 0);
    k_pack_e4m3<<<(unsigned)((n1 + 255) / 256), 256, 0, st>>>((const uint8_t*)u, dst, I, H, 1, 0);
    k_pack_e4m3<<<(unsigned)((n2 + 255) / 256), 256, 0, st>>>((const uint8_t*)dn, dst, H, I, 2, p2_off);
    const int P1 = I / kTileRows, P2 = H / (2 * kTileRows);
    k_scale_tables<<<P1 + P2, 2, 0, st>>>(sg, su, sd, reinterpret_cast<float*>(dst + (size_t)3 * H * I), P1, P2, H / 128, I / 128);
  }
}

// Once per step, before the first expert launch: the fp16 copy of x the e4m3 path contracts with.
void caee_launch_umma_prepare(caee_ctx* c, const void* x, int T, cudaStream_t st) {
  if (c->d.w_dtype != CAEE_E4M3 || T <= 0) return;
  caee_launch_fp8_prepare(c, x, T, st);
  return;
  const size_t n = (size_t)T * c->d.H;
  k_bf16_to_f16<<<(unsigned)((n / 2 + 256) / 256), 256, 0, st>>>((const __nv_bfloat16*)x, c->x16, n);
}

// runs [run_begin, run_begin + run_count) (run_count < 0: every run of the work list), tile
// tickets from wl.sched[ticket].
void caee_launch_expert_umma(caee_ctx* c, const void* x, int T, int run_begin, int run_count, int ticket, cudaStream_t st) {
  const caee_layer_desc& d = c->d;
  const bool fp8 = d.w_dtype == CAEE_E4M3;
  if (fp8) {
    caee_launch_expert_fp8(c, T, run_begin, run_count, ticket, st);
    return;
  }
  UmmaParams p;
  p.wl = c->wl;
  p.packed = c->packed.dev_ptrs;
  p.x = fp8 ? (const uint16_t*)c->x16 : (const uint16_t*)x;  // fp8: caee_launch_umma_prepare widened x
  p.hbuf = (uint16_t*)c->hbuf_b16;
  p.obuf = c->obuf;
  p.H = d.H; p.I = d.I;
  p.P1 = d.I / kTileRows; p.P2 = d.H / (2 * kTileRows);
  p.KB1 = d.H / kKBlock; p.KB2 = d.I / kKBlock;
  p.run_begin = run_begin; p.run_count = run_count; p.ticket = ticket;
  p.sc_off = (int)((size_t)3 * d.H * d.I);
  p.r2_off = p.P1 * (d.H / 128) * 2 + p.P1 * 2;
  const int ncap = std::min(CAEE_RUN_TOKENS, (T + 15) & ~15);
  p.b_stage_bytes = ncap * kKBlock * 2;
  p.stage_bytes = kAStageBytes + p.b_stage_bytes;
  const int max_dyn = 227 * 1024 - 6144;            // leave room for the static barriers / ratio block
  const int smem_budget = max_dyn - 1024;           // alignment slack
  size_t dyn;
  if (fp8) {
    p.n_stages = 4;
    p.n_land = std::min(kMaxStages, (smem_budget - p.n_stages * p.stage_bytes) / kLandBytes);
    if (p.n_land < 4) { p.n_stages = 3; p.n_land = std::min(kMaxStages, (smem_budget - p.n_stages * p.stage_bytes) / kLandBytes); }
    p.land_off = p.n_stages * p.stage_bytes;
    dyn = (size_t)p.land_off + (size_t)p.n_land * kLandBytes + 1024;
  } else {
    p.n_stages = std::min(kMaxStages, smem_budget / p.stage_bytes);
    p.n_land = 0; p.land_off = 0;
    dyn = (size_t)p.n_stages * p.stage_bytes + 1024;
  }
  static bool attr_set = false;
  if (!attr_set) {
    cudaFuncSetAttribute(k_expert_umma<false>, cudaFuncAttributeMaxDynamicSharedMemorySize, max_dyn);
    cudaFuncSetAttribute(k_expert_umma<true>, cudaFuncAttributeMaxDynamicSharedMemorySize, max_dyn);
    attr_set = true;
  }
  if (fp8) k_expert_umma<true><<<c->num_sms, kThreadsFp8, dyn, st>>>(p);
  else k_expert_umma<false><<<c->num_sms, kThreads, dyn, st>>>(p);
}
