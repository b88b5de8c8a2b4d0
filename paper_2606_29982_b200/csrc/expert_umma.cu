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
// Roles (256 threads, 1 CTA per SM):  warp 0 = weight producer (one lane issues bulk copies),
// warp 1 = MMA issuer (one lane), warps 2-3 = token-operand loaders (warp 2 also owns TMEM
// alloc/free), warps 4-7 = epilogue (TMEM -> registers -> SwiGLU -> h, or -> o rows).
// Tiles are claimed dynamically (one atomic ticket per tile, phase-1 tickets first); a
// phase-2 tile only waits (per-run counter) for phase-1 tiles, which never wait, so the
// schedule cannot deadlock and CTAs that finish early simply claim more tiles.
#include "caee_internal.cuh"

namespace {

constexpr int kThreads = 256;
constexpr int kTileRows = 128;          // UMMA M
constexpr int kKBlock = 64;             // k elements per stage
constexpr int kATileBytes = kTileRows * kKBlock * 2;  // 16 KB
constexpr int kAStageBytes = 2 * kATileBytes;         // 32 KB: two tiles per stage
constexpr int kTmemCols = 512;
constexpr int kMaxStages = 8;

struct UmmaParams {
  caee_worklist wl;
  uint8_t* const* packed;     // [E+S] stage images
  const __nv_bfloat16* x;     // [T,H]
  __nv_bfloat16* hbuf;        // [rows,I]
  float* obuf;                // [T*(k+S),H]
  int H, I;
  int P1, P2, KB1, KB2;       // tiles per run and k-blocks per tile, per phase
  int n_stages, b_stage_bytes, stage_bytes;
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
// kind::f16 instruction descriptor: D fp32, A/B bf16, both K-major, M = 128, N = n.
__device__ __forceinline__ uint32_t make_idesc(int n) {
  return (1u << 4) | (1u << 7) | (1u << 10) | ((uint32_t)(n >> 3) << 17) | ((uint32_t)(kTileRows >> 4) << 24);
}

__device__ __forceinline__ int ld_acquire(const int* p) {
  int v;
  asm volatile("ld.acquire.gpu.global.s32 %0, [%1];" : "=r"(v) : "l"(p) : "memory");
  return v;
}
struct Tile {
  int phase, run, sub;  // sub = ft (phase 1) or op (phase 2)
};
__device__ __forceinline__ bool tile_at(int i, int n_runs, int P1, int P2, Tile& t) {
  const int t1 = n_runs * P1;
  if (i < t1) { t.phase = 1; t.run = i / P1; t.sub = i - t.run * P1; return true; }
  i -= t1;
  if (i < n_runs * P2) { t.phase = 2; t.run = i / P2; t.sub = i - t.run * P2; return true; }
  return false;
}

// ------------------------------------------------------------------ the kernel
constexpr int kQueue = 4;      // tile-queue depth (producer runs at most this many tiles ahead)
constexpr int kLag = 3;        // token-operand stages each loader warp keeps in flight (cp.async groups)

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

__global__ void __launch_bounds__(kThreads, 1) k_expert_umma(const UmmaParams p) {
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
  const int n_runs = p.wl.meta[1];

  if (threadIdx.x == 0) {
    for (int s = 0; s < p.n_stages; ++s) {
      mbar_init(full0 + 8 * s, 3);   // producer's expect_tx arrive + 2 loader warps
      mbar_init(empty0 + 8 * s, 1);  // tcgen05.commit
    }
    for (int a = 0; a < 2; ++a) {
      mbar_init(tfull0 + 8 * a, 1);   // tcgen05.commit
      mbar_init(tempty0 + 8 * a, 4);  // one lane of each epilogue warp
    }
    for (int q = 0; q < kQueue; ++q) {
      mbar_init(qfull0 + 8 * q, 1);   // producer
      mbar_init(qempty0 + 8 * q, 7);  // MMA warp + 2 loader warps + 4 epilogue warps
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

  if (warp == 0) {
    // ===== weight producer: claims tiles; one 32 KB bulk copy per stage from the packed image
    if (lane == 0) {
      int stage = 0, ph = 0, q = 0, qph = 0;
      for (;;) {
        mbar_wait(qempty0 + 8 * q, qph ^ 1);
        const int i = atomicAdd(p.wl.sched, 1);
        tq_slots[q] = i;
        mbar_arrive(qfull0 + 8 * q);
        if (++q == kQueue) { q = 0; qph ^= 1; }
        if (!tile_at(i, n_runs, p.P1, p.P2, t)) break;
        const int e = p.wl.run_expert[t.run];
        const int nkb = t.phase == 1 ? p.KB1 : p.KB2;
        const uint8_t* src = p.packed[e] + (t.phase == 1 ? (size_t)t.sub * p.KB1 : (size_t)p.P1 * p.KB1 + (size_t)t.sub * p.KB2) * kAStageBytes;
        for (int kb = 0; kb < nkb; ++kb) {
          mbar_wait(empty0 + 8 * stage, ph ^ 1);
          mbar_arrive_expect_tx(full0 + 8 * stage, kAStageBytes);
          bulk_g2s(smem_base + stage * p.stage_bytes, src + (size_t)kb * kAStageBytes, kAStageBytes, full0 + 8 * stage);
          if (++stage == p.n_stages) { stage = 0; ph ^= 1; }
        }
      }
    }
  } else if (warp == 1) {
    // ===== MMA issuer (the whole warp pops the queue; one lane issues)
    int stage = 0, ph = 0;
    for (int it = 0; tile_at(tq.pop(), n_runs, p.P1, p.P2, t); ++it) {
      if (lane == 0) {
        const int as = it & 1;
        const int npad = (p.wl.run_n[t.run] + 15) & ~15;
        const uint32_t idesc = make_idesc(npad);
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
    auto publish = [&](int count) {  // the oldest `count` in-flight stages have landed
      fence_proxy_async_smem();
      __syncwarp();
      for (int j = 0; j < count; ++j) {
        if (lane == 0) mbar_arrive(full0 + 8 * pend_stage);
        if (++pend_stage == p.n_stages) pend_stage = 0;
      }
      pending -= count;
    };
    while (tile_at(tq.pop(), n_runs, p.P1, p.P2, t)) {
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
          const int* flag = p.wl.sched + 2 + t.run;
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
        if (pending > kLag) {
          asm volatile("cp.async.wait_group %0;" ::"n"(kLag) : "memory");
          publish(1);
        }
      }
      // flush at the tile boundary: nothing of this tile may wait behind a later tile's dependency
      asm volatile("cp.async.wait_group 0;" ::: "memory");
      publish(pending);
    }
  } else {
    // ===== epilogue: TMEM -> registers -> SwiGLU -> h (phase 1) or -> o rows (phase 2)
    const int q = warp - 4;  // TMEM lane quadrant of this warp (warp % 4)
    for (int it = 0; tile_at(tq.pop(), n_runs, p.P1, p.P2, t); ++it) {
      const int as = it & 1;
      const int n = p.wl.run_n[t.run], start = p.wl.run_start[t.run];
      mbar_wait(tfull0 + 8 * as, (it >> 1) & 1);
      tc_fence_after();
      const uint32_t tbase = tmem_base + ((uint32_t)(q * 32) << 16) + as * 256;
      const int row = q * 32 + lane;
      if (t.phase == 1) {
        __nv_bfloat16* hcol = p.hbuf + (size_t)p.wl.run_hrow[t.run] * p.I + t.sub * kTileRows + row;
        for (int c = 0; c < n; c += 16) {
          uint32_t g[16], u[16];
          tmem_ld16(tbase + c, g);
          tmem_ld16(tbase + 128 + c, u);
          tmem_ld_wait();
#pragma unroll
          for (int j = 0; j < 16; ++j) {
            if (c + j < n) {
              const float gv = __uint_as_float(g[j]), uv = __uint_as_float(u[j]);
              hcol[(size_t)(c + j) * p.I] = __float2bfloat16_rn(gv / (1.0f + __expf(-gv)) * uv);
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
        // publish this tile's slice of h: all 128 epilogue threads' stores, then one release add
        __threadfence();
        asm volatile("bar.sync 1, 128;" ::: "memory");
        if (threadIdx.x == 128) atomicAdd(p.wl.sched + 2 + t.run, 1);
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
  if (d.w_dtype != CAEE_BF16 || d.act_dtype != CAEE_BF16) {
    *why = "the UMMA expert kernel takes bf16 weights and bf16 activations";
    return CAEE_EDTYPE;
  }
  if (d.H % 256 || d.I % 128) {
    *why = "the UMMA expert kernel needs H % 256 == 0 and I % 128 == 0";
    return CAEE_ESHAPE;
  }
  return CAEE_OK;
}

size_t caee_umma_packed_bytes(const caee_ctx* c) { return (size_t)3 * c->d.H * c->d.I * 2; }

void caee_launch_pack_expert(caee_ctx* c, int e, uint8_t* dst, const void* g, const void* u, const void* dn, const float*,
                             const float*, const float*, cudaStream_t st) {
  (void)e;
  const int H = c->d.H, I = c->d.I;
  const size_t n1 = (size_t)I * (H / 8), n2 = (size_t)H * (I / 8);
  const size_t p2_off = (size_t)2 * I * H * 2;
  k_pack_bf16<<<(unsigned)((n1 + 255) / 256), 256, 0, st>>>((const __nv_bfloat16*)g, dst, I, H, 0, 0);
  k_pack_bf16<<<(unsigned)((n1 + 255) / 256), 256, 0, st>>>((const __nv_bfloat16*)u, dst, I, H, 1, 0);
  k_pack_bf16<<<(unsigned)((n2 + 255) / 256), 256, 0, st>>>((const __nv_bfloat16*)dn, dst, H, I, 2, p2_off);
}

void caee_launch_expert_umma(caee_ctx* c, const void* x, int T, cudaStream_t st) {
  const caee_layer_desc& d = c->d;
  UmmaParams p;
  p.wl = c->wl;
  p.packed = c->packed.dev_ptrs;
  p.x = (const __nv_bfloat16*)x;
  p.hbuf = c->hbuf_b16;
  p.obuf = c->obuf;
  p.H = d.H; p.I = d.I;
  p.P1 = d.I / kTileRows; p.P2 = d.H / (2 * kTileRows);
  p.KB1 = d.H / kKBlock; p.KB2 = d.I / kKBlock;
  const int ncap = std::min(CAEE_RUN_TOKENS, (T + 15) & ~15);
  p.b_stage_bytes = ncap * kKBlock * 2;
  p.stage_bytes = kAStageBytes + p.b_stage_bytes;
  const int max_dyn = 227 * 1024 - 4096;            // leave room for the static barriers block
  const int smem_budget = max_dyn - 1024;           // alignment slack
  p.n_stages = std::min(kMaxStages, smem_budget / p.stage_bytes);
  const size_t dyn = (size_t)p.n_stages * p.stage_bytes + 1024;
  static bool attr_set = false;
  if (!attr_set) {
    cudaFuncSetAttribute(k_expert_umma, cudaFuncAttributeMaxDynamicSharedMemorySize, max_dyn);
    attr_set = true;
  }
  k_expert_umma<<<c->num_sms, kThreads, dyn, st>>>(p);
}
