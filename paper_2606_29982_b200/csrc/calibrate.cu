// calibrate.cu — S10 offline calibration: "a brief offline profiling
// phase" that fits  C~(e,d) = alpha_d * S_e / B_d + beta_d  for the two data-movement tiers
// of this box: streaming reads from HBM, and pinned-host -> device copies over PCIe.
// Each tier is timed at several transfer sizes with CUDA events; t = slope*S + intercept
// is fitted by ordinary least squares (slope = alpha_d/B_d, intercept = beta_d).
#include <algorithm>
#include <cmath>

#include "caee_internal.cuh"

namespace {

// Streams `n16` 16-byte words and keeps the loads alive through a never-true store.
__global__ void __launch_bounds__(256) k_stream_read(const uint4* __restrict__ src, size_t n16, unsigned* __restrict__ sink) {
  unsigned acc = 0;
  const size_t stride = (size_t)gridDim.x * blockDim.x;
  size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
  for (; i + 3 * stride < n16; i += 4 * stride) {
    uint4 a, b, c, d;
    asm volatile("ld.global.nc.L1::no_allocate.v4.u32 {%0,%1,%2,%3}, [%4];" : "=r"(a.x), "=r"(a.y), "=r"(a.z), "=r"(a.w) : "l"(src + i));
    asm volatile("ld.global.nc.L1::no_allocate.v4.u32 {%0,%1,%2,%3}, [%4];" : "=r"(b.x), "=r"(b.y), "=r"(b.z), "=r"(b.w) : "l"(src + i + stride));
    asm volatile("ld.global.nc.L1::no_allocate.v4.u32 {%0,%1,%2,%3}, [%4];" : "=r"(c.x), "=r"(c.y), "=r"(c.z), "=r"(c.w) : "l"(src + i + 2 * stride));
    asm volatile("ld.global.nc.L1::no_allocate.v4.u32 {%0,%1,%2,%3}, [%4];" : "=r"(d.x), "=r"(d.y), "=r"(d.z), "=r"(d.w) : "l"(src + i + 3 * stride));
    acc ^= a.x ^ a.y ^ a.z ^ a.w ^ b.x ^ b.y ^ b.z ^ b.w ^ c.x ^ c.y ^ c.z ^ c.w ^ d.x ^ d.y ^ d.z ^ d.w;
  }
  for (; i < n16; i += stride) {
    uint4 a;
    asm volatile("ld.global.nc.L1::no_allocate.v4.u32 {%0,%1,%2,%3}, [%4];" : "=r"(a.x), "=r"(a.y), "=r"(a.z), "=r"(a.w) : "l"(src + i));
    acc ^= a.x ^ a.y ^ a.z ^ a.w;
  }
  if (acc == 0x9e3779b9u) *sink = acc;
}

bool ols(const std::vector<double>& S, const std::vector<double>& t, caee_cost_fit* f) {
  const int n = (int)S.size();
  if (n < 2) return false;
  double ms = 0, mt = 0;
  for (int i = 0; i < n; ++i) { ms += S[i]; mt += t[i]; }
  ms /= n; mt /= n;
  double sxx = 0, sxy = 0, syy = 0;
  for (int i = 0; i < n; ++i) { sxx += (S[i] - ms) * (S[i] - ms); sxy += (S[i] - ms) * (t[i] - mt); syy += (t[i] - mt) * (t[i] - mt); }
  if (sxx <= 0) return false;
  f->slope_ns_per_byte = sxy / sxx;
  f->intercept_ns = mt - f->slope_ns_per_byte * ms;
  double sse = 0;
  for (int i = 0; i < n; ++i) { double r = t[i] - (f->slope_ns_per_byte * S[i] + f->intercept_ns); sse += r * r; }
  f->r2 = syy > 0 ? 1.0 - sse / syy : 1.0;
  f->gbytes_per_s = f->slope_ns_per_byte > 0 ? 1.0 / f->slope_ns_per_byte : 0.0;
  f->n_points = n;
  f->valid = f->slope_ns_per_byte > 0;
  return f->valid != 0;
}

double median(std::vector<float>& v) {
  std::sort(v.begin(), v.end());
  return v[v.size() / 2];
}

}  // namespace

caee_status caee_calibrate_impl(caee_ctx* c, const caee_calib_opts* o, caee_cost_fit fit[2]) {
  const caee_layer_desc& d = c->d;
  const int64_t expert_bytes = 3LL * d.H * d.I * (d.w_dtype == CAEE_F32 ? 4 : d.w_dtype == CAEE_BF16 ? 2 : 1);
  int n_sizes = (o && o->n_sizes) ? o->n_sizes : 6;
  int iters = (o && o->iters) ? o->iters : 10;
  int64_t lo = (o && o->min_bytes) ? o->min_bytes : (4LL << 20);
  int64_t hi = (o && o->max_bytes) ? o->max_bytes : std::max<int64_t>(expert_bytes, 8LL << 20);
  if (n_sizes < 2 || n_sizes > 16 || iters < 1 || iters > 1000 || lo < 4096 || hi <= lo || hi > (4LL << 30))
    return caee_fail(c, CAEE_EINVAL, "bad calibration options");
  memset(fit, 0, sizeof(caee_cost_fit) * 2);
  for (int t = 0; t < 2; ++t) { c->calib_bytes[t].clear(); c->calib_ns[t].clear(); }
  std::vector<int64_t> sizes(n_sizes);
  for (int i = 0; i < n_sizes; ++i) {
    double f = (double)i / (n_sizes - 1);
    sizes[i] = ((int64_t)std::llround((double)lo * std::pow((double)hi / (double)lo, f)) + 4095) & ~4095LL;
  }
  sizes[n_sizes - 1] = (hi + 4095) & ~4095LL;
  const int64_t l2_guard = 512LL << 20;  // pool much larger than L2 so every timed read comes from HBM
  const int64_t pool_bytes = l2_guard + sizes.back();
  uint8_t* pool = nullptr;
  unsigned* sink = nullptr;
  uint8_t* hostbuf = nullptr;
  cudaEvent_t e0 = nullptr, e1 = nullptr;
  cudaStream_t st = nullptr;
  caee_status rc = CAEE_OK;
#define CK(expr) do { cudaError_t _e = (expr); if (_e != cudaSuccess) { rc = caee_check_cuda(c, _e, #expr); goto done; } } while (0)
  CK(cudaMalloc((void**)&pool, pool_bytes));
  CK(cudaMalloc((void**)&sink, 4));
  CK(cudaMemset(pool, 1, pool_bytes));
  CK(cudaEventCreate(&e0));
  CK(cudaEventCreate(&e1));
  CK(cudaStreamCreateWithFlags(&st, cudaStreamNonBlocking));
  {
    // tier 0: HBM streaming reads
    std::vector<double> S, Tm;
    const int grid = c->num_sms * 8;
    int64_t off = 0;
    for (int64_t sz : sizes) {
      std::vector<float> ms;
      for (int it = 0; it < iters + 2; ++it) {
        if (off + sz > pool_bytes) off = 0;
        CK(cudaEventRecord(e0, st));
        k_stream_read<<<grid, 256, 0, st>>>(reinterpret_cast<const uint4*>(pool + off), (size_t)sz / 16, sink);
        CK(cudaEventRecord(e1, st));
        CK(cudaEventSynchronize(e1));
        float t;
        CK(cudaEventElapsedTime(&t, e0, e1));
        if (it >= 2) ms.push_back(t);
        off += (sz + 4095) & ~4095LL;
      }
      S.push_back((double)sz);
      Tm.push_back(median(ms) * 1e6);
    }
    ols(S, Tm, &fit[0]);
    c->calib_bytes[0] = S; c->calib_ns[0] = Tm;
  }
  {
    // tier 1: pinned host -> device copies (the paper's H2D transfer of a cache-miss expert)
    cudaError_t he = cudaMallocHost((void**)&hostbuf, sizes.back());
    if (he != cudaSuccess) {
      cudaGetLastError();
      fit[1].valid = 0;
    } else {
      memset(hostbuf, 1, sizes.back());
      std::vector<double> S, Tm;
      for (int64_t sz : sizes) {
        std::vector<float> ms;
        for (int it = 0; it < iters + 1; ++it) {
          CK(cudaEventRecord(e0, st));
          CK(cudaMemcpyAsync(pool, hostbuf, sz, cudaMemcpyHostToDevice, st));
          CK(cudaEventRecord(e1, st));
          CK(cudaEventSynchronize(e1));
          float t;
          CK(cudaEventElapsedTime(&t, e0, e1));
          if (it >= 1) ms.push_back(t);
        }
        S.push_back((double)sz);
        Tm.push_back(median(ms) * 1e6);
      }
      ols(S, Tm, &fit[1]);
      c->calib_bytes[1] = S; c->calib_ns[1] = Tm;
    }
  }
done:
#undef CK
  if (hostbuf) cudaFreeHost(hostbuf);
  if (pool) cudaFree(pool);
  if (sink) cudaFree(sink);
  if (e0) cudaEventDestroy(e0);
  if (e1) cudaEventDestroy(e1);
  if (st) cudaStreamDestroy(st);
  if (rc == CAEE_OK && !fit[0].valid) rc = caee_fail(c, CAEE_ECUDA, "HBM tier calibration produced no valid fit");
  return rc;
}
