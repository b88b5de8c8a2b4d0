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
// B operand (tokens): x rows (phase 1) or h rows (phase 2), 128 bytes (64 k) per row and stage,
// gathered by the TMA unit (cp.async.bulk.tensor tile::gather4: four rows per instruction, rows
// named by the work list, padding rows zero-filled) into 128-byte-swizzled 8-row atoms — the
// SWIZZLE_128B K-major layout the token-operand descriptor names.
//
// e4m3 weights have their own kernel (expert_fp8.cu).
//
// Roles (256 threads; 1 CTA per SM):  warp 0 = weight producer (one lane issues bulk copies),
// warp 1 = MMA issuer (one lane), warp 2 = token-operand loader (one TMA gather per lane and stage; also owns TMEM
// alloc/free), warps 4-7 = epilogue (TMEM -> registers -> SwiGLU -> h, or -> o rows).
// Tiles are claimed dynamically (one atomic ticket per tile, phase-1 tickets first); a
// phase-2 tile only waits (per-run counter) for phase-1 tiles, which never wait, so the
// schedule cannot deadlock and CTAs that finish early simply claim more tiles.
#include <cstring>

#include "umma_common.cuh"

namespace {

using namespace caee_umma;

constexpr int kThreads = 256;
constexpr int kKBlock = 64;             // k elements per stage

struct UmmaParams {
  caee_worklist wl;
  uint8_t* const* packed;     // [E+S] stage images
  const uint16_t* x;          // [T,H] bf16
  uint16_t* hbuf;             // [rows,I] bf16
  float* obuf;                // [T*(k+S),H]
  int H, I;
  int P1, P2, KB1, KB2;       // tiles per run and 64-k stages per tile, per phase
  int n_stages, b_stage_bytes, stage_bytes;
  int run_begin, run_count;   // runs [run_begin, run_begin + run_count) of the work list; run_count < 0: all
  int ticket;                 // which tile-ticket counter of wl.sched this launch uses
  CUtensorMap tm_x, tm_h;     // byte maps over x [T, 2H] and hbuf [rows, 2I] for the TMA row gathers
  KSplit ksp;                 // split k range of phase-1 tiles in steps of a few tokens (umma_common.cuh)
};

// ------------------------------------------------------------------ the kernel
__global__ void __launch_bounds__(kThreads, 1) k_expert_umma(const __grid_constant__ UmmaParams p) {
  extern __shared__ __align__(1024) uint8_t smem_raw[];
  uint8_t* smem = reinterpret_cast<uint8_t*>((reinterpret_cast<uintptr_t>(smem_raw) + 1023) & ~(uintptr_t)1023);
  __shared__ __align__(8) uint64_t bars[2 * kMaxStages + 4 + 2 * kQueue];
  __shared__ uint32_t tmem_base_s;
  __shared__ int tq_slots[kQueue];

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
      mbar_init(tfull0 + 8 * a, 1);   // tcgen05.commit
      mbar_init(tempty0 + 8 * a, 4);  // one lane of each epilogue warp
    }
    for (int q = 0; q < kQueue; ++q) {
      mbar_init(qfull0 + 8 * q, 1);                // producer
      mbar_init(qempty0 + 8 * q, 6);               // MMA warp + loader warp + 4 epilogue warps
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
  // everything above touched only shared memory and TMEM: with a programmatic dependent launch it
  // overlaps the decision kernel's tail; the work list exists from here on
  griddep_wait();
  griddep_launch();
  const int n_runs = p.run_count >= 0 ? p.run_count : p.wl.meta[1];
  const int KS = (p.ksp.ks > 1 && n_runs * p.P1 <= p.ksp.tile_cap) ? p.ksp.ks : 1;
  const TileMap tm{n_runs, p.run_begin, p.P1, p.P2, KS};
  const int KB1s = p.KB1 / KS;             // 64-k stages of one phase-1 (sub-)tile
  TileQueue tq{qfull0, qempty0, tq_slots, 0, 0};
  Tile t;

  if (warp == 0) {
    // ===== weight producer: claims tiles; one bulk copy per stage from the packed image
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
        nxt = (int)gridDim.x + atomicAdd(p.wl.sched + p.ticket, 1);
        for (int kb = 0; kb < nkb; ++kb) {
          mbar_wait(empty0 + 8 * stage, ph ^ 1);
          mbar_arrive_expect_tx(full0 + 8 * stage, kAStageBytes);
          bulk_g2s_stream(smem_base + stage * p.stage_bytes, src + (size_t)kb * kAStageBytes, kAStageBytes, full0 + 8 * stage, pol);
          if (++stage == p.n_stages) { stage = 0; ph ^= 1; }
          if (kb == (nkb >> 1)) {
            vn = tm.at(nxt, tn);
            if (vn) resolve(tn, srcn, nkbn);
          }
        }
      }
    }
  } else if (warp == 1) {
    // ===== MMA issuer: the whole warp runs the loop (uniform control flow keeps the descriptor
    // arithmetic on the uniform datapath); one elected lane issues
    int stage = 0, ph = 0;
    for (int it = 0; tm.at(tq.pop(), t); ++it) {
      const int as = it & 1;
      const int npad = (__shfl_sync(0xffffffffu, p.wl.run_n[t.run], 0) + 15) & ~15;
      const uint32_t idesc = make_idesc(npad, true);
      const int nkb = t.phase == 1 ? KB1s : p.KB2;
      mbar_wait(tempty0 + 8 * as, ((it >> 1) & 1) ^ 1);
      const uint32_t d0 = tmem_base + as * 256, d1 = d0 + 128;
      for (int kb = 0; kb < nkb; ++kb) {
        mbar_wait(full0 + 8 * stage, ph);
        tc_fence_after();
        const uint32_t a_addr = smem_base + stage * p.stage_bytes;
        const uint64_t a0 = make_desc(a_addr), a1 = make_desc(a_addr + kATileBytes), b = make_desc_sw128(a_addr + kAStageBytes);
        if (elect_one()) {
          if (kb == 0) {
            umma_bf16_imm<false>(d0, a0, b, idesc);
            umma_bf16_imm<false>(d1, a1, b, idesc);
          } else {
            umma_bf16_imm<true>(d0, a0, b, idesc);
            umma_bf16_imm<true>(d1, a1, b, idesc);
          }
#pragma unroll
          for (int ks = 1; ks < kKBlock / 16; ++ks) {   // per 16-element k-step: weights +256 B, tokens +32 B (>> 4)
            umma_bf16_imm<true>(d0, a0 + (uint64_t)(ks * 16), b + (uint64_t)(ks * 2), idesc);
            umma_bf16_imm<true>(d1, a1 + (uint64_t)(ks * 16), b + (uint64_t)(ks * 2), idesc);
          }
          tc_commit(empty0 + 8 * stage);
          if (kb == nkb - 1) tc_commit(tfull0 + 8 * as);
        }
        __syncwarp();
        if (++stage == p.n_stages) { stage = 0; ph ^= 1; }
      }
    }
  } else if (warp == 2) {
    // ===== token-operand loader: TMA row gathers (tile::gather4: 4 rows x 128 B per instruction)
    // of the x rows (phase 1) or h rows (phase 2) of the run into 128-byte-swizzled 8-row atoms;
    // lane l owns rows 4l..4l+3, padding rows come back as zeros
    int stage = 0, ph = 0;
    while (tm.at(tq.pop(), t)) {
      const int n = p.wl.run_n[t.run], start = p.wl.run_start[t.run];
      const int npad = (n + 15) & ~15;
      const int nkb = t.phase == 1 ? KB1s : p.KB2, kb0 = t.kq * KB1s;     // kq = 0 in phase 2
      const CUtensorMap* tmap = t.phase == 1 ? &p.tm_x : &p.tm_h;
      int r[4];
#pragma unroll
      for (int i = 0; i < 4; ++i) {
        const int row = lane * 4 + i;
        r[i] = kOobRow;
        if (row < n) r[i] = t.phase == 1 ? p.wl.ent_tok[start + row] : p.wl.run_hrow[t.run] + row;
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
        if (lane == 0) mbar_arrive_expect_tx(full0 + 8 * stage, (uint32_t)npad * 128u);
        __syncwarp();
        if (mine) tma_gather4(b_addr + lane * 512, tmap, full0 + 8 * stage, (kb0 + kb) * 128, r[0], r[1], r[2], r[3]);
        if (++stage == p.n_stages) { stage = 0; ph ^= 1; }
      }
    }
  } else if (warp == 3) {
    // ===== reducer (only in steps that split their phase-1 tiles, KSplit): finishes tiles whose ks
    // partial sums are complete; lane l holds features 4 l .. 4 l + 3
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
          const uint32_t w0 = (uint32_t)__bfloat16_as_ushort(__float2bfloat16_rn(h0)) | ((uint32_t)__bfloat16_as_ushort(__float2bfloat16_rn(h1)) << 16);
          const uint32_t w1 = (uint32_t)__bfloat16_as_ushort(__float2bfloat16_rn(h2)) | ((uint32_t)__bfloat16_as_ushort(__float2bfloat16_rn(h3)) << 16);
          *reinterpret_cast<uint2*>(p.hbuf + (size_t)(hrow + c) * p.I + ft * kTileRows + 4 * lane) = make_uint2(w0, w1);
        }
        // publish the tile's slice of h (read through the async proxy by other SMs' TMA gathers)
        asm volatile("fence.proxy.async;" ::: "memory");
        __threadfence();
        __syncwarp();
        if (lane == 0) atomicAdd(p.wl.ready + run, 1);
      }
    }
  } else if (warp < 8) {
    // ===== epilogue: TMEM -> registers -> SwiGLU -> h (phase 1) or -> o rows (phase 2)
    const int q = warp - 4;  // TMEM lane quadrant of this warp (warp % 4)
    for (int it = 0; tm.at(tq.pop(), t); ++it) {
      const int as = it & 1;
      const int n = p.wl.run_n[t.run], start = p.wl.run_start[t.run];
      mbar_wait(tfull0 + 8 * as, (it >> 1) & 1);
      tc_fence_after();
      const uint32_t tbase = tmem_base + ((uint32_t)(q * 32) << 16) + as * 256;
      const int row = q * 32 + lane;
      if (t.phase == 1 && KS > 1) {
        // split k range (KSplit, umma_common.cuh): leave this sub-tile's partial sums and count it; a
        // reducer warp finishes the tile (n <= kKSplitCols)
        uint32_t g[8], u[8];
        tmem_ld8(tbase, g);
        tmem_ld8(tbase + 128, u);
        tmem_ld_wait();
        tc_fence_before();
        __syncwarp();
        if (lane == 0) mbar_arrive(tempty0 + 8 * as);
        const int tile = (t.run - p.run_begin) * p.P1 + t.sub;
        CAEE_DEV_ASSERT(tile >= 0 && tile < p.ksp.tile_cap && n <= kKSplitCols);
        float* mine = p.ksp.part + ((size_t)tile * KS + t.kq) * (2 * kKSplitCols * kTileRows);
#pragma unroll
        for (int c = 0; c < kKSplitCols; ++c) {
          if (c < n) {
            __stcg(mine + c * kTileRows + row, __uint_as_float(g[c]));
            __stcg(mine + (kKSplitCols + c) * kTileRows + row, __uint_as_float(u[c]));
          }
        }
        asm volatile("bar.sync 2, 128;" ::: "memory");
        if (threadIdx.x == 128) {
          __threadfence();                      // cumulative: the CTA's partial stores, ordered by the barrier
          atomicAdd(p.ksp.cnt + tile, 1);
        }
        continue;
      }
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
              const float gv = __uint_as_float(g[j]), uv = __uint_as_float(u[j]);
              const float hv = gv / (1.0f + __expf(-gv)) * uv;
              hcol[(size_t)(c + j) * p.I] = __bfloat16_as_ushort(__float2bfloat16_rn(hv));
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
              CAEE_DEV_ASSERT(p.wl.ent_dst[start + c + j] >= 0 && p.wl.ent_dst[start + c + j] < p.wl.ent_cap);
              float* o = caee_o_base(p.wl, p.obuf, p.wl.ent_tok[start + c + j]) + (ocol - p.obuf) + (size_t)p.wl.ent_dst[start + c + j] * p.H;
              o[0] = __uint_as_float(d0[j]);
              o[kTileRows] = __uint_as_float(d1[j]);
            }
          }
        }
      }
      tc_fence_before();
      __syncwarp();
      if (lane == 0) mbar_arrive(tempty0 + 8 * as);
      if (t.phase == 1) {
        // publish this tile's slice of h: all 128 epilogue threads' stores (read later through the
        // async proxy by other SMs' TMA gathers), then one release add
        asm volatile("fence.proxy.async;" ::: "memory");
        __threadfence();
        asm volatile("bar.sync 1, 128;" ::: "memory");
        if (threadIdx.x == 128) atomicAdd(p.wl.ready + t.run, 1);
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

}  // namespace

caee_status caee_umma_supported(const caee_ctx* c, std::string* why) {
  const caee_layer_desc& d = c->d;
  if ((d.w_dtype != CAEE_BF16 && d.w_dtype != CAEE_E4M3) || d.act_dtype != CAEE_BF16) {
    *why = "the UMMA expert kernels take bf16 or e4m3 weights and bf16 activations";
    return CAEE_EDTYPE;
  }
  if (d.H % 256 || d.I % 128) {
    *why = "the UMMA expert kernels need H % 256 == 0 and I % 128 == 0";
    return CAEE_ESHAPE;
  }
  if (d.w_dtype == CAEE_E4M3) return caee_fp8_supported(c, why);
  return CAEE_OK;
}

size_t caee_umma_packed_bytes(const caee_ctx* c) {
  if (c->d.w_dtype == CAEE_E4M3) return caee_fp8_packed_bytes(c);
  return (size_t)3 * c->d.H * c->d.I * 2;
}

void caee_launch_pack_expert(caee_ctx* c, int e, uint8_t* dst, const void* g, const void* u, const void* dn, const float* sg,
                             const float* su, const float* sd, cudaStream_t st) {
  (void)e;
  const int H = c->d.H, I = c->d.I;
  if (c->d.w_dtype == CAEE_E4M3) {
    caee_launch_pack_expert_fp8(c, dst, g, u, dn, sg, su, sd, st);
    return;
  }
  const size_t n1 = (size_t)I * (H / 8), n2 = (size_t)H * (I / 8);
  const size_t p2_off = (size_t)2 * I * H * 2;
  k_pack_bf16<<<(unsigned)((n1 + 255) / 256), 256, 0, st>>>((const __nv_bfloat16*)g, dst, I, H, 0, 0);
  k_pack_bf16<<<(unsigned)((n1 + 255) / 256), 256, 0, st>>>((const __nv_bfloat16*)u, dst, I, H, 1, 0);
  k_pack_bf16<<<(unsigned)((n2 + 255) / 256), 256, 0, st>>>((const __nv_bfloat16*)dn, dst, H, I, 2, p2_off);
}

// Once per step, before the first expert launch (e4m3: x -> its two e4m3 terms, expert_fp8.cu).
void caee_launch_umma_prepare(caee_ctx* c, const void* x, int T, cudaStream_t st) {
  if (c->d.w_dtype != CAEE_E4M3) return;
  if (c->step_prefill) caee_launch_fp8_wide_prepare(c, x, T, st);
  else caee_launch_fp8_prepare(c, x, T, st);
}

// runs [run_begin, run_begin + run_count) (run_count < 0: every run of the work list), tile
// tickets from wl.sched[ticket].
caee_status caee_launch_expert_umma(caee_ctx* c, const void* x, int T, int run_begin, int run_count, int ticket, cudaStream_t st) {
  const caee_layer_desc& d = c->d;
  if (d.w_dtype == CAEE_E4M3) {
    if (c->step_prefill == 2) caee_launch_expert_fp8_ts(c, T, run_begin, run_count, ticket, st);
    else if (c->step_prefill == 1) caee_launch_expert_fp8_wide(c, T, run_begin, run_count, ticket, st);
    else caee_launch_expert_fp8(c, T, run_begin, run_count, ticket, st);
    return CAEE_OK;
  }
  ++c->n_launches;
  UmmaParams p;
  p.wl = c->wl;
  p.packed = c->packed.dev_ptrs;
  p.x = (const uint16_t*)x;
  p.hbuf = (uint16_t*)c->hbuf_b16;
  p.obuf = c->obuf;
  p.H = d.H; p.I = d.I;
  p.P1 = d.I / kTileRows; p.P2 = d.H / (2 * kTileRows);
  p.KB1 = d.H / kKBlock; p.KB2 = d.I / kKBlock;
  p.run_begin = run_begin; p.run_count = run_count; p.ticket = ticket;
  // x is the caller's buffer: its map is encoded per call (host-side, ~1 us); h is ours
  if (!c->tm_ready) {
    if (!encode_row_gather_map(c->tm_h, c->hbuf_b16, (size_t)d.I * 2, c->h_rows_cap))
      return caee_fail(c, CAEE_ECUDA, "cuTensorMapEncodeTiled failed for the h scratch");
    c->tm_ready = true;
  }
  if (!encode_row_gather_map(&p.tm_x, x, (size_t)d.H * 2, (size_t)T))
    return caee_fail(c, CAEE_EINVAL, "cuTensorMapEncodeTiled refused x (it must be 16-byte aligned device memory)");
  memcpy(&p.tm_h, c->tm_h, sizeof(CUtensorMap));
  const int ncap = std::min((int)c->wl.run_cap, (T + 15) & ~15);
  p.b_stage_bytes = ncap * kKBlock * 2;
  p.stage_bytes = kAStageBytes + p.b_stage_bytes;
  const int max_dyn = 227 * 1024 - 4096;            // leave room for the static barriers
  p.n_stages = std::min(kMaxStages, (max_dyn - 1024) / p.stage_bytes);
  const size_t dyn = (size_t)p.n_stages * p.stage_bytes + 1024;
  p.ksp = caee_ksplit_for(c, T, p.KB1, ticket);
  if (!(c->attr_done & 1u)) {
    cudaFuncSetAttribute(k_expert_umma, cudaFuncAttributeMaxDynamicSharedMemorySize, max_dyn);
    c->attr_done |= 1u;
  }
  if (c->pdl && !c->any_offload) {
    // programmatic dependent launch: the CTAs are scheduled while the decision kernel still runs
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = dim3((unsigned)c->num_sms);
    cfg.blockDim = dim3(kThreads);
    cfg.dynamicSmemBytes = dyn;
    cfg.stream = st;
    cudaLaunchAttribute at[1];
    at[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    at[0].val.programmaticStreamSerializationAllowed = 1;
    cfg.attrs = at; cfg.numAttrs = 1;
    cudaLaunchKernelEx(&cfg, k_expert_umma, p);
    return CAEE_OK;
  }
  k_expert_umma<<<c->num_sms, kThreads, dyn, st>>>(p);
  return CAEE_OK;
}
