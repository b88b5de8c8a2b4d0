// router_mma.cu — S0 router logits on the tensor cores for steps of >= 64 tokens (router
// form per DESIGN.md reading R1): partial[ks][t][e] = sum_{h in chunk ks} x[t,h] W_r[e,h].
//
// Why.  At 4096 tokens the router is a 15 GFLOP dense contraction; on fp32 FMAs (router.cu) it took
// 0.49 ms of a 4.9 ms step (here 45 us), and 31 us of a 128-token decode step (here 14 us).  The scores decide integers (top-k picks), so the contraction has to keep
// fp32 accuracy: W_r (fp32) is split ONCE, at caee_set_router, into three bf16 terms
//     w = hi + mid + lo,   hi = bf16(w), mid = bf16(w - hi), lo = bf16(w - hi - mid)     (exact: 3 x 8 bits)
// and x is bf16 already, so every product x * term is exact in fp32 and the tensor core adds them into
// fp32 accumulators in TMEM: the only rounding left is the accumulation's, as on the FMA path.
// Three tcgen05.mma kind::f16 passes (45 GFLOP in bf16) cost ~40 us.
//
// Shape.  CTA (mt, ks): tokens [128 mt, +128) x all E experts (N = E <= 256, one MMA tile) x the
// k range of split ks, in 64-k stages.  A = the x tile, fetched by ONE tiled TMA load per stage
// (128 rows x 128 B, 128-byte swizzle; rows beyond T come back as zeros); B = the three W_r terms of
// the stage, pre-packed by k_pack_router in the UMMA canonical K-major no-swizzle order (8 rows x 16 B
// core matrices; LBO 128 B, SBO 1024 B), ONE bulk copy of 3 E 128 bytes per stage.  The CTA writes its
// fp32 partial tile; the consumer (caee_token_scores, warp_select.cuh) adds a token's partials in
// ascending ks — a fixed order, deterministic scores.
//
// Roles (192 threads): warp 0 = producer (one lane), warp 1 = MMA issuer (owns TMEM), warps 2-5 =
// epilogue (TMEM lane quadrant = warp % 4).
#include <cstring>

#include "umma_common.cuh"

namespace {

using namespace caee_umma;

constexpr int kThreads = 192;
constexpr int kKStage = 64;                    // k per stage
constexpr int kXTileBytes = 128 * kKStage * 2; // 16 KB: 128 tokens x 64 k
constexpr int kRingMax = 6;
constexpr int kTmemRouterCols = 256;

struct RouterMmaParams {
  CUtensorMap tm_x;        // x [T, H] bf16, box 64 x 128, 128-byte swizzle
  const uint8_t* wimg;     // [H/64][3][E rows x 64 k] bf16 terms of W_r (k_pack_router)
  float* partial;          // [ksplit][T][E]
  int T, E;
  int n_stage_total, sps;  // H / 64; stages per split
  int n_ring, stage_bytes, w_term_bytes;
};

__global__ void __launch_bounds__(kThreads, 1) k_router_mma(const __grid_constant__ RouterMmaParams p) {
  extern __shared__ __align__(1024) uint8_t smem_raw[];
  uint8_t* smem = reinterpret_cast<uint8_t*>((reinterpret_cast<uintptr_t>(smem_raw) + 1023) & ~(uintptr_t)1023);
  __shared__ __align__(8) uint64_t bars[2 * kRingMax + 1];
  __shared__ uint32_t tmem_base_s;
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const uint32_t smem_base = smem_u32(smem);
  const uint32_t full0 = smem_u32(&bars[0]), empty0 = smem_u32(&bars[kRingMax]), tfull = smem_u32(&bars[2 * kRingMax]);
  const int mt = blockIdx.x, ks = blockIdx.y;
  const int s_lo = ks * p.sps, s_hi = min(p.n_stage_total, s_lo + p.sps);

  if (threadIdx.x == 0) {
    for (int s = 0; s < p.n_ring; ++s) {
      mbar_init(full0 + 8 * s, 1);    // the producer's expect_tx arrive
      mbar_init(empty0 + 8 * s, 1);   // tcgen05.commit
    }
    mbar_init(tfull, 1);
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
  }
  if (warp == 1) {
    asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], %1;" ::"r"(smem_u32(&tmem_base_s)), "n"(kTmemRouterCols));
    asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;");
  }
  tc_fence_before();
  __syncthreads();
  tc_fence_after();
  const uint32_t tmem_base = tmem_base_s;

  if (warp == 0) {
    if (lane == 0) {
      int st = 0, ph = 0;
      const uint32_t tx = (uint32_t)kXTileBytes + 3u * (uint32_t)p.w_term_bytes;
      for (int s = s_lo; s < s_hi; ++s) {
        mbar_wait(empty0 + 8 * st, ph ^ 1);
        mbar_arrive_expect_tx(full0 + 8 * st, tx);
        const uint32_t dst = smem_base + st * p.stage_bytes;
        tma_tile_2d(dst, &p.tm_x, full0 + 8 * st, s * kKStage, mt * 128);
        bulk_g2s(dst + kXTileBytes, p.wimg + (size_t)s * 3 * p.w_term_bytes, 3u * (uint32_t)p.w_term_bytes, full0 + 8 * st);
        if (++st == p.n_ring) { st = 0; ph ^= 1; }
      }
    }
  } else if (warp == 1) {
    // whole warp in the loop (uniform control flow), one elected lane issues
    int st = 0, ph = 0;
    const uint32_t idesc = make_idesc(p.E, true);
    for (int s = s_lo; s < s_hi; ++s) {
      mbar_wait(full0 + 8 * st, ph);
      tc_fence_after();
      const uint32_t a_addr = smem_base + st * p.stage_bytes;
      const uint64_t a = make_desc_sw128(a_addr);
      if (elect_one()) {
#pragma unroll
        for (int term = 0; term < 3; ++term) {
          const uint64_t b = make_desc(a_addr + kXTileBytes + term * p.w_term_bytes);
#pragma unroll
          for (int k16 = 0; k16 < kKStage / 16; ++k16) {   // per 16-k step: x +32 B (>> 4), W +256 B
            if (s == s_lo && term == 0 && k16 == 0) umma_bf16_imm<false>(tmem_base, a, b, idesc);
            else umma_bf16_imm<true>(tmem_base, a + (uint64_t)(k16 * 2), b + (uint64_t)(k16 * 16), idesc);
          }
        }
        tc_commit(empty0 + 8 * st);
        if (s == s_hi - 1) tc_commit(tfull);
      }
      __syncwarp();
      if (++st == p.n_ring) { st = 0; ph ^= 1; }
    }
  } else {
    // epilogue: thread = one token row (TMEM lane), 16 expert columns per load
    const int q = warp & 3, row = q * 32 + lane, t = mt * 128 + row;
    if (s_hi > s_lo) {
      mbar_wait(tfull, 0);
      tc_fence_after();
    }
    float* out = p.partial + ((size_t)ks * p.T + (size_t)min(t, p.T - 1)) * p.E;
    const uint32_t taddr = tmem_base + ((uint32_t)(q * 32) << 16);
    for (int c = 0; c < p.E; c += 16) {
      uint32_t v[16];
      if (s_hi > s_lo) {
        tmem_ld16(taddr + c, v);
        tmem_ld_wait();
      } else {
#pragma unroll
        for (int j = 0; j < 16; ++j) v[j] = 0u;
      }
      if (t < p.T) {
#pragma unroll
        for (int j = 0; j < 16; j += 4)
          *reinterpret_cast<uint4*>(out + c + j) = make_uint4(v[j], v[j + 1], v[j + 2], v[j + 3]);
      }
    }
  }
  tc_fence_before();
  __syncthreads();
  if (warp == 1) {
    tc_fence_after();
    asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;" ::"r"(tmem_base), "n"(kTmemRouterCols));
  }
}

// W_r [E, H] fp32 -> stage images of its three bf16 terms.  One thread per (expert, 8-k chunk).
__global__ void __launch_bounds__(256) k_pack_router(const float* __restrict__ Wr, uint8_t* __restrict__ img, int E, int H) {
  const size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
  const int cpr = H / 8;
  if (i >= (size_t)E * cpr) return;
  const int e = (int)(i / cpr), k0 = (int)(i % cpr) * 8;
  const int s = k0 / kKStage, c = (k0 % kKStage) / 8;
  const float4 a = *reinterpret_cast<const float4*>(Wr + (size_t)e * H + k0);
  const float4 b = *reinterpret_cast<const float4*>(Wr + (size_t)e * H + k0 + 4);
  const float w[8] = {a.x, a.y, a.z, a.w, b.x, b.y, b.z, b.w};
  uint16_t t[3][8];
#pragma unroll
  for (int j = 0; j < 8; ++j) {
    const __nv_bfloat16 hi = __float2bfloat16_rn(w[j]);
    const float r1 = w[j] - __bfloat162float(hi);
    const __nv_bfloat16 mid = __float2bfloat16_rn(r1);
    const float r2 = r1 - __bfloat162float(mid);
    const __nv_bfloat16 lo = __float2bfloat16_rn(r2);
    t[0][j] = __bfloat16_as_ushort(hi); t[1][j] = __bfloat16_as_ushort(mid); t[2][j] = __bfloat16_as_ushort(lo);
  }
  const size_t term_bytes = (size_t)E * kKStage * 2;
#pragma unroll
  for (int term = 0; term < 3; ++term) {
    uint8_t* dst = img + ((size_t)s * 3 + term) * term_bytes + (size_t)(e / 8) * 1024 + c * 128 + (e % 8) * 16;
    *reinterpret_cast<uint4*>(dst) = make_uint4((uint32_t)t[term][0] | ((uint32_t)t[term][1] << 16), (uint32_t)t[term][2] | ((uint32_t)t[term][3] << 16),
                                                (uint32_t)t[term][4] | ((uint32_t)t[term][5] << 16), (uint32_t)t[term][6] | ((uint32_t)t[term][7] << 16));
  }
}

}  // namespace

// bf16 activations, E a multiple of 16 up to 256 (one MMA N tile), H a multiple of 64
bool caee_router_mma_supported(const caee_ctx* c) {
  const caee_layer_desc& d = c->d;
  return d.act_dtype == CAEE_BF16 && d.E % 16 == 0 && d.E >= 16 && d.E <= 256 && d.H % kKStage == 0;
}

size_t caee_router_mma_image_bytes(const caee_ctx* c) { return (size_t)3 * c->d.E * c->d.H * 2; }

bool caee_router_uses_mma(const caee_ctx* c, int T) { return c->wr_img != nullptr && T >= c->router_mma_min_tokens; }

// split-K of the MMA router for a T-token step: about one CTA per SM, at least 4 stages per split
void caee_router_mma_shape(const caee_ctx* c, int T, int* ksplit, int* sps) {
  const int n_stage = c->d.H / kKStage, m_tiles = caee_ceil_div(T, 128);
  int ks = std::max(1, c->num_sms / m_tiles);
  ks = std::min(ks, std::max(1, n_stage / 4));
  const int per = caee_ceil_div(n_stage, ks);
  *ksplit = caee_ceil_div(n_stage, per);
  if (sps) *sps = per;
}

void caee_launch_pack_router(caee_ctx* c, cudaStream_t st) {
  const size_t n = (size_t)c->d.E * (c->d.H / 8);
  k_pack_router<<<(unsigned)((n + 255) / 256), 256, 0, st>>>(c->Wr, c->wr_img, c->d.E, c->d.H);
}

caee_status caee_launch_router_mma(caee_ctx* c, const void* x, int T, cudaStream_t st) {
  const caee_layer_desc& d = c->d;
  RouterMmaParams p;
  if (!encode_tile_map_bf16(&p.tm_x, x, (size_t)T, (size_t)d.H, 128))
    return caee_fail(c, CAEE_EINVAL, "cuTensorMapEncodeTiled refused x (it must be 16-byte aligned device memory)");
  p.wimg = c->wr_img;
  p.partial = c->partial;
  p.T = T; p.E = d.E;
  p.n_stage_total = d.H / kKStage;
  int ks;
  caee_router_mma_shape(c, T, &ks, &p.sps);
  p.w_term_bytes = d.E * kKStage * 2;
  p.stage_bytes = kXTileBytes + 3 * p.w_term_bytes;
  const int max_dyn = 227 * 1024 - 2048;
  p.n_ring = std::min(kRingMax, (max_dyn - 1024) / p.stage_bytes);
  const size_t dyn = (size_t)p.n_ring * p.stage_bytes + 1024;
  if (!(c->attr_done & 8u)) {
    cudaFuncSetAttribute(k_router_mma, cudaFuncAttributeMaxDynamicSharedMemorySize, max_dyn);
    c->attr_done |= 8u;
  }
  ++c->n_launches;
  k_router_mma<<<dim3((unsigned)caee_ceil_div(T, 128), (unsigned)ks), kThreads, dyn, st>>>(p);
  return CAEE_OK;
}
