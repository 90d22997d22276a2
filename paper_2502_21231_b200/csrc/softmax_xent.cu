// softmax_xent.cu — bs_softmax_xent: fused softmax cross-entropy ("fuses numerous
// operations into a single kernel, takes BF16 inputs, and still performs online computations in
// FP32 precision").  Per token: loss = logsumexp(x) - x[label], dlogits = g (softmax(x) - onehot).
//
// HBM-bound: every logit is read once and every gradient written once (2 + 2 bytes per element).
// A block owns one row at a time: pass A streams the row from HBM with 128-bit loads into shared
// memory while each thread keeps an online (max, sum) pair in fp32; after the block reduction
// pass B re-reads the row from shared memory, not from HBM, and streams the gradients out.  Rows
// of V <= kMaxSmemV logits take this path (V/TP = 16K at the paper's 128K vocabulary and TP = 8
// is 32 KB, so several blocks per SM overlap one row's loads with another row's stores); longer
// rows read the logits a second time from global memory (mostly L2).
#include <cuda_bf16.h>
#include <cuda_runtime.h>
#include <math_constants.h>

#include <algorithm>

#include "common.h"
#include "launch_utils.h"
#include "ptx.cuh"

namespace {

constexpr int kThreads = 256;
#ifndef BS_XENT_BLOCKS8
#define BS_XENT_BLOCKS8 3  // resident blocks per SM of the 16K-logit register kernel
#endif
constexpr int kMaxSmemV = 48 * 1024;  // 96 KB of bf16: two blocks per SM

struct XentParams {
  const __nv_bfloat16* logits;
  const int32_t* labels;
  float* loss;
  __nv_bfloat16* dlogits;
  int64_t row_stride;  // elements, logits and dlogits
  int32_t n_tokens, vocab;
  float grad_scale;
};

__device__ __forceinline__ uint4 ldg_stream(const uint4* p) {
  uint4 r;
  asm volatile("ld.global.nc.L1::no_allocate.v4.u32 {%0,%1,%2,%3}, [%4];"
               : "=r"(r.x), "=r"(r.y), "=r"(r.z), "=r"(r.w)
               : "l"(p));
  return r;
}
__device__ __forceinline__ void stg_stream(uint4* p, const uint4& v) {
  asm volatile("st.global.L1::no_allocate.v4.u32 [%0], {%1,%2,%3,%4};" ::"l"(p), "r"(v.x),
               "r"(v.y), "r"(v.z), "r"(v.w)
               : "memory");
}
__device__ __forceinline__ float lo(uint32_t u) { return __uint_as_float(u << 16); }
__device__ __forceinline__ float hi(uint32_t u) { return __uint_as_float(u & 0xffff0000u); }
__device__ __forceinline__ uint32_t pack2(float a, float b) {
  __nv_bfloat162 t = __floats2bfloat162_rn(a, b);
  return *reinterpret_cast<uint32_t*>(&t);
}

using bs::ptx::add2;
using bs::ptx::ex2;
using bs::ptx::fma2;
using bs::ptx::fmax3;
using bs::ptx::mul2;

// running (max, sum of exp(x - max)) over 8 more logits; base-2 exponentials (one MUFU each),
// packed fp32x2 arithmetic around them: the kernel is HBM-bound only as long as it issues few
// instructions per logit (~3.5 in each pass)
__device__ __forceinline__ void online8(const uint4& v, float& m, float2& l) {
  constexpr float kLog2e = 1.4426950408889634f;
  const uint32_t u[4] = {v.x, v.y, v.z, v.w};
  float mx = m;
#pragma unroll
  for (int i = 0; i < 4; ++i) mx = fmax3(mx, lo(u[i]), hi(u[i]));
  if (mx > m) {  // (-inf - finite) * log2e = -inf -> 2^-inf = 0 at the first chunk
    const float a = ex2((m - mx) * kLog2e);
    l = mul2(l, make_float2(a, a));
    m = mx;
  }
  const float nm = -m * kLog2e;
  const float2 nm2 = make_float2(nm, nm), k2 = make_float2(kLog2e, kLog2e);
#pragma unroll
  for (int i = 0; i < 4; ++i) {
    const float2 t = fma2(make_float2(lo(u[i]), hi(u[i])), k2, nm2);
    l = add2(l, make_float2(ex2(t.x), ex2(t.y)));
  }
}

template <bool kSmemRow>
__global__ void __launch_bounds__(kThreads) softmax_xent_kernel(const XentParams p) {
  extern __shared__ __align__(16) uint8_t smem_raw[];
  uint4* row_s = reinterpret_cast<uint4*>(smem_raw);
  __shared__ float red_m[kThreads / 32], red_l[kThreads / 32];
  __shared__ float row_lse;
  constexpr float kLog2e = 1.4426950408889634f;
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  const int nvec = p.vocab >> 3;          // whole 8-logit vectors
  const int tail0 = nvec << 3;            // first logit of the ragged tail (vocab % 8 != 0)
  for (int row = blockIdx.x; row < p.n_tokens; row += gridDim.x) {
    const __nv_bfloat16* x = p.logits + (int64_t)row * p.row_stride;
    __nv_bfloat16* dx = p.dlogits + (int64_t)row * p.row_stride;
    const int label = p.labels[row];
    const uint4* xv = reinterpret_cast<const uint4*>(x);
    uint4* dv = reinterpret_cast<uint4*>(dx);
    if (label < 0) {  // ignored token: no loss, zero gradient (block-uniform branch)
      for (int i = tid; i < nvec; i += kThreads) stg_stream(dv + i, make_uint4(0, 0, 0, 0));
      for (int j = tail0 + tid; j < p.vocab; j += kThreads) dx[j] = __float2bfloat16(0.f);
      if (tid == 0) p.loss[row] = 0.f;
      continue;
    }
    // ---- pass A: stream the row in, online max / sum per thread ----
    float m = -CUDART_INF_F;
    float2 l2 = make_float2(0.f, 0.f);
    int i = tid;
    for (; i + 3 * kThreads < nvec; i += 4 * kThreads) {  // four loads in flight per thread
      uint4 v[4];
#pragma unroll
      for (int k = 0; k < 4; ++k) v[k] = ldg_stream(xv + i + k * kThreads);
#pragma unroll
      for (int k = 0; k < 4; ++k) {
        if (kSmemRow) row_s[i + k * kThreads] = v[k];
        online8(v[k], m, l2);
      }
    }
    for (; i < nvec; i += kThreads) {
      const uint4 v = ldg_stream(xv + i);
      if (kSmemRow) row_s[i] = v;
      online8(v, m, l2);
    }
    float l = l2.x + l2.y;
    for (int j = tail0 + tid; j < p.vocab; j += kThreads) {
      const float f = __bfloat162float(x[j]);
      if (f > m) {
        l *= exp2f((m - f) * kLog2e);
        m = f;
      }
      l += exp2f((f - m) * kLog2e);
    }
    // ---- block reduction of (m, l) ----
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
      const float m2 = __shfl_xor_sync(0xffffffffu, m, o), l2 = __shfl_xor_sync(0xffffffffu, l, o);
      const float mx = fmaxf(m, m2);
      // a thread that saw no logit has (m, l) = (-inf, 0): its term is 0, not NaN
      l = (m == mx ? l : l * exp2f((m - mx) * kLog2e)) + (m2 == mx ? l2 : l2 * exp2f((m2 - mx) * kLog2e));
      m = mx;
    }
    if (lane == 0) {
      red_m[warp] = m;
      red_l[warp] = l;
    }
    __syncthreads();  // also: the row is complete in shared memory
    if (warp == 0) {
      m = lane < kThreads / 32 ? red_m[lane] : -CUDART_INF_F;
      l = lane < kThreads / 32 ? red_l[lane] : 0.f;
#pragma unroll
      for (int o = 4; o > 0; o >>= 1) {
        const float m2 = __shfl_xor_sync(0xffffffffu, m, o), l2 = __shfl_xor_sync(0xffffffffu, l, o);
        const float mx = fmaxf(m, m2);
        l = (m == mx ? l : l * exp2f((m - mx) * kLog2e)) + (m2 == mx ? l2 : l2 * exp2f((m2 - mx) * kLog2e));
        m = mx;
      }
      if (lane == 0) {
        const float lse = m + logf(l);
        row_lse = lse;
        p.loss[row] = lse - __bfloat162float(x[label]);
      }
    }
    __syncthreads();
    // ---- pass B: gradients g (exp(x - lse) - onehot), from shared memory ----
    const float nl = -row_lse * kLog2e, g = p.grad_scale;
    const float2 nl2 = make_float2(nl, nl), k2 = make_float2(kLog2e, kLog2e), g2 = make_float2(g, g);
    const int lab_vec = label >> 3, lab_sub = label & 7;
    for (int i2 = tid; i2 < nvec; i2 += kThreads) {
      const uint4 v = kSmemRow ? row_s[i2] : ldg_stream(xv + i2);
      const uint32_t u[4] = {v.x, v.y, v.z, v.w};
      float2 e[4];
#pragma unroll
      for (int k = 0; k < 4; ++k) {
        const float2 t = fma2(make_float2(lo(u[k]), hi(u[k])), k2, nl2);
        e[k] = make_float2(ex2(t.x), ex2(t.y));
      }
      if (i2 == lab_vec) {
#pragma unroll
        for (int k = 0; k < 4; ++k) {
          if (2 * k == lab_sub) e[k].x -= 1.f;
          if (2 * k + 1 == lab_sub) e[k].y -= 1.f;
        }
      }
      uint32_t w[4];
#pragma unroll
      for (int k = 0; k < 4; ++k) {
        const float2 d = mul2(e[k], g2);
        w[k] = pack2(d.x, d.y);
      }
      stg_stream(dv + i2, make_uint4(w[0], w[1], w[2], w[3]));
    }
    for (int j = tail0 + tid; j < p.vocab; j += kThreads) {
      float e = exp2f(fmaf(__bfloat162float(x[j]), kLog2e, nl));
      if (j == label) e -= 1.f;
      dx[j] = __float2bfloat16(e * g);
    }
    __syncthreads();  // the next row overwrites row_s / row_lse
  }
}

// Rows of at most kThreads * 8 * kVpt logits (16K at kVpt = 8: V / TP of the paper's example):
// the whole row lives in the registers of the block - packed bf16 while the maximum is taken,
// then fp32 exponentials - so that every logit costs ONE exponential (the MUFU unit of B200
// delivers 16 per clock and SM; with two per logit it, not HBM, set the time) and no shared
// memory traffic at all.  The vocab % 8 tail logits go through thread 0's scalar path.
template <int kVpt>
__global__ void __launch_bounds__(kThreads, kVpt >= 8 ? BS_XENT_BLOCKS8 : 6)
softmax_xent_reg_kernel(const XentParams p) {
  __shared__ float red[2][kThreads / 32];
  constexpr float kLog2e = 1.4426950408889634f;
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  const int nvec = p.vocab >> 3, tail0 = nvec << 3;
  const float2 k2 = make_float2(kLog2e, kLog2e);
  auto block_reduce = [&](float v, bool is_max, int buf) {
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
      const float w = __shfl_xor_sync(0xffffffffu, v, o);
      v = is_max ? fmaxf(v, w) : v + w;
    }
    if (lane == 0) red[buf][warp] = v;
    __syncthreads();
    v = red[buf][0];
#pragma unroll
    for (int w = 1; w < kThreads / 32; ++w) v = is_max ? fmaxf(v, red[buf][w]) : v + red[buf][w];
    return v;
  };
  for (int row = blockIdx.x; row < p.n_tokens; row += gridDim.x) {
    const __nv_bfloat16* x = p.logits + (int64_t)row * p.row_stride;
    __nv_bfloat16* dx = p.dlogits + (int64_t)row * p.row_stride;
    const int label = p.labels[row];
    const uint4* xv = reinterpret_cast<const uint4*>(x);
    uint4* dv = reinterpret_cast<uint4*>(dx);
    if (label < 0) {  // ignored token (block-uniform branch)
      for (int i = tid; i < nvec; i += kThreads) stg_stream(dv + i, make_uint4(0, 0, 0, 0));
      for (int j = tail0 + tid; j < p.vocab; j += kThreads) dx[j] = __float2bfloat16(0.f);
      if (tid == 0) p.loss[row] = 0.f;
      continue;
    }
    // all loads of the row in flight at once
    uint4 v[kVpt];
#pragma unroll
    for (int k = 0; k < kVpt; ++k) {
      const int i = tid + k * kThreads;
      v[k] = i < nvec ? ldg_stream(xv + i) : make_uint4(0xff80ff80u, 0xff80ff80u, 0xff80ff80u, 0xff80ff80u);
    }  // (0xff80 = bf16 -inf: no contribution to the maximum or the sum)
    float m = -CUDART_INF_F;
#pragma unroll
    for (int k = 0; k < kVpt; ++k) {
      const uint32_t u[4] = {v[k].x, v[k].y, v[k].z, v[k].w};
#pragma unroll
      for (int q = 0; q < 4; ++q) m = fmax3(m, lo(u[q]), hi(u[q]));
    }
    if (tid == 0)
      for (int j = tail0; j < p.vocab; ++j) m = fmaxf(m, __bfloat162float(x[j]));
    m = block_reduce(m, true, 0);
    // exponentials, once per logit, kept in registers
    const float nm = -m * kLog2e;
    const float2 nm2 = make_float2(nm, nm);
    float2 e[kVpt][4];
    float2 l2 = make_float2(0.f, 0.f);
#pragma unroll
    for (int k = 0; k < kVpt; ++k) {
      const uint32_t u[4] = {v[k].x, v[k].y, v[k].z, v[k].w};
#pragma unroll
      for (int q = 0; q < 4; ++q) {
        const float2 t = fma2(make_float2(lo(u[q]), hi(u[q])), k2, nm2);
        e[k][q] = make_float2(ex2(t.x), ex2(t.y));
        l2 = add2(l2, e[k][q]);
      }
    }
    float l = l2.x + l2.y;
    if (tid == 0)
      for (int j = tail0; j < p.vocab; ++j) l += ex2(fmaf(__bfloat162float(x[j]), kLog2e, nm));
    l = block_reduce(l, false, 1);
    const float lse = m + logf(l);
    if (tid == 0) p.loss[row] = lse - __bfloat162float(x[label]);
    // gradients g (e / l - onehot)
    const float s = p.grad_scale / l;
    const float2 s2 = make_float2(s, s);
    const int lab_vec = label >> 3, lab_sub = label & 7;
#pragma unroll
    for (int k = 0; k < kVpt; ++k) {
      const int i = tid + k * kThreads;
      if (i < nvec) {
        uint32_t w[4];
#pragma unroll
        for (int q = 0; q < 4; ++q) {
          float2 d = mul2(e[k][q], s2);
          if (i == lab_vec) {
            if (2 * q == lab_sub) d.x -= p.grad_scale;
            if (2 * q + 1 == lab_sub) d.y -= p.grad_scale;
          }
          w[q] = pack2(d.x, d.y);
        }
        stg_stream(dv + i, make_uint4(w[0], w[1], w[2], w[3]));
      }
    }
    if (tid == 0)
      for (int j = tail0; j < p.vocab; ++j) {
        float d = ex2(fmaf(__bfloat162float(x[j]), kLog2e, nm)) * s;
        if (j == label) d -= p.grad_scale;
        dx[j] = __float2bfloat16(d);
      }
    // (red[0] / red[1] are rewritten only behind the next row's barriers: no barrier needed here)
  }
}

template <int kVpt>
void launch_reg(const XentParams& p, int sms, cudaStream_t st) {
  const int per_sm = kVpt >= 8 ? BS_XENT_BLOCKS8 : 6;
  const int grid = std::min(p.n_tokens, sms * per_sm);
  softmax_xent_reg_kernel<kVpt><<<grid, kThreads, 0, st>>>(p);
}

}  // namespace

extern "C" bs_status_t bs_softmax_xent(const void* logits, const int32_t* labels, int32_t n_tokens,
                                       int32_t vocab, int64_t row_stride, float grad_scale,
                                       float* loss, void* dlogits, void* stream) {
  BS_REQUIRE(n_tokens >= 0 && vocab >= 1, BS_ERR_INVALID_ARG,
             "bs_softmax_xent: n_tokens %d, vocab %d", n_tokens, vocab);
  BS_REQUIRE(row_stride >= vocab && row_stride % 8 == 0, BS_ERR_INVALID_ARG,
             "bs_softmax_xent: row_stride %lld must be >= vocab and a multiple of 8 elements",
             (long long)row_stride);
  if (n_tokens == 0) return BS_OK;
  BS_REQUIRE(logits && labels && loss && dlogits, BS_ERR_INVALID_ARG,
             "bs_softmax_xent: null pointer");
  BS_REQUIRE((((uintptr_t)logits | (uintptr_t)dlogits) & 15) == 0, BS_ERR_INVALID_ARG,
             "bs_softmax_xent: logits and dlogits must be 16-byte aligned");
  cudaStream_t st = (cudaStream_t)stream;
  bs_status_t rc = bs::check_device();
  if (rc != BS_OK) return rc;
  const int sms = bs::sm_count();
  XentParams p{(const __nv_bfloat16*)logits, labels, loss, (__nv_bfloat16*)dlogits, row_stride,
               n_tokens, vocab, grad_scale};
  const int nvec = vocab / 8;
  if (nvec <= kThreads * 2) {
    launch_reg<2>(p, sms, st);
  } else if (nvec <= kThreads * 4) {
    launch_reg<4>(p, sms, st);
  } else if (nvec <= kThreads * 8) {
    launch_reg<8>(p, sms, st);
  } else if (vocab <= kMaxSmemV) {
    const size_t smem = (size_t)(vocab / 8) * 16;
    const int per_sm = (int)std::max<size_t>(1, std::min<size_t>(8, (200 * 1024) / (smem + 1024)));
    rc = bs::set_max_smem_once((const void*)softmax_xent_kernel<true>, kMaxSmemV * 2, 4);
    if (rc != BS_OK) return rc;
    const int grid = std::min(n_tokens, sms * per_sm);
    softmax_xent_kernel<true><<<grid, kThreads, smem, st>>>(p);
  } else {
    const int grid = std::min(n_tokens, sms * 8);
    softmax_xent_kernel<false><<<grid, kThreads, 0, st>>>(p);
  }
  bs::count_launch();
  BS_CUDA(cudaGetLastError());
  return BS_OK;
}
