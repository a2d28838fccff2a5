// NEXT-4: the consumer of the hot path -- GraphSAGE (mean aggregator) forward, loss, backward and
// SGD over the sampled blocks and the gathered feature tensor (Alg. 1 l.15).
//
// One warp per destination row; lane l owns the columns l, l+32, l+64, l+96 of the row (dims <= 128).
//   k_sage_fwd   self row + mean of the neighbor rows in registers (the feature tensor is read once,
//                row-contiguous 128-byte segments), then the two small products against weights
//                held TRANSPOSED in shared memory (lane-consecutive columns: no bank conflicts);
//                writes agg (kept for the backward pass) and the activated output
//   k_sage_loss  one thread per seed: softmax cross-entropy, its gradient, per-seed loss
//   k_sage_wgrad parameter gradients as a skinny reduction over the rows (register accumulators,
//                coalesced reads of h_in / agg, g tiles in shared memory)
//   k_sage_bwd   (layers > 0) the gradient of the layer's input: activation mask, the two small
//                products against the transposed weights, scattered through the mean with float atomics
//   k_sage_sgd   p -= lr * g, g = 0
// Nothing here is a large dense contraction (hidden size 16): the step is bound by the gather-like
// reads of the aggregation, not by tensor-core work.
#include <algorithm>
#include <vector>

#include "common.cuh"
#include "kernels.h"

namespace gg {

constexpr int kSageWarps = 8;
constexpr int kSlotsIn = 4;    // columns per lane, input side  (dims <= 128)
constexpr int kSlotsOut = 2;   // columns per lane, output side (dims <= 64)
constexpr int kSageMaxFeatureDim = 1024;   // first layer's input, walked in slabs of 128 columns

__device__ __forceinline__ float warp_sum(float v) {
#pragma unroll
  for (int o = 16; o; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
  return v;
}

// one halving step of the reduce-scatter butterfly: N values stay, N go to the partner lane
template <int N, int OFF>
__device__ __forceinline__ void bfly(float (&p)[16], int lane) {
  const bool hi = (lane & OFF) != 0;
#pragma unroll
  for (int k = 0; k < N; ++k) {
    const float send = hi ? p[k] : p[k + N];
    const float keepv = hi ? p[k + N] : p[k];
    p[k] = keepv + __shfl_xor_sync(0xffffffffu, send, OFF);
  }
}

template <bool RELU>
__global__ void __launch_bounds__(2 * kSageWarps * 32, 2)   // 8 warps per CTA, 16 when the weights fill the SM's shared memory
k_sage_fwd(const float* __restrict__ h_in, const int32_t* __restrict__ indptr,
           const int32_t* __restrict__ src_local, int n_dst, int din, int dout,
           const float* __restrict__ w_self, const float* __restrict__ w_neigh,
           const float* __restrict__ bias, float* __restrict__ agg_out, float* __restrict__ h_out) {
  extern __shared__ float s_w[];   // two weight matrices (layout below), then [dout] bias
  // dout <= 16: rows of 17 floats per input column ([c][17]: odd pitch, lane-consecutive columns hit
  // distinct banks and output o is an immediate offset); otherwise transposed [o][din]
  const bool narrow = dout <= 16;
  const int wsize = narrow ? 17 * din : dout * din;
  float* ws = s_w;
  float* wn = s_w + wsize;
  float* sb = wn + wsize;
  for (int k = threadIdx.x; k < din * dout; k += blockDim.x) {
    const int c = k / dout, o = k - c * dout;
    const int at = narrow ? c * 17 + o : o * din + c;
    ws[at] = w_self[k];
    wn[at] = w_neigh[k];
  }
  for (int k = threadIdx.x; k < dout; k += blockDim.x) sb[k] = bias[k];
  __syncthreads();
  const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5, nw = blockDim.x >> 5;
  for (int i = blockIdx.x * nw + wid; i < n_dst; i += gridDim.x * nw) {
    const int e0 = indptr[i], e1 = indptr[i + 1];
    const float deg = (float)(e1 - e0);
    float p[16];
#pragma unroll
    for (int o = 0; o < 16; ++o) p[o] = 0.0f;
    float xs[kSlotsIn], ac[kSlotsIn];
    // input columns in slabs of 128 (4 per lane); a feature row wider than 128 (the paper's Reddit
    // shape, 602) walks the row's neighbor list once per slab and keeps the 16 partial outputs
    for (int c0 = 0; c0 < din; c0 += 32 * kSlotsIn) {
#pragma unroll
      for (int s = 0; s < kSlotsIn; ++s) {
        const int c = c0 + lane + 32 * s;
        xs[s] = c < din ? h_in[(int64_t)i * din + c] : 0.0f;
        ac[s] = 0.0f;
      }
      for (int eb = e0; eb < e1; eb += 32) {
        // 32 neighbor ids at a time, then their rows back to back (independent loads)
        const int mine = eb + lane < e1 ? __ldg(src_local + eb + lane) : 0;
        const int cnt = min(32, e1 - eb);
#pragma unroll 4
        for (int q = 0; q < cnt; ++q) {
          const int64_t src = __shfl_sync(0xffffffffu, mine, q);
#pragma unroll
          for (int s = 0; s < kSlotsIn; ++s) {
            const int c = c0 + lane + 32 * s;
            if (c < din) ac[s] += __ldg(h_in + src * din + c);
          }
        }
      }
#pragma unroll
      for (int s = 0; s < kSlotsIn; ++s) {
        const int c = c0 + lane + 32 * s;
        ac[s] = (e1 > e0 && c < din) ? ac[s] / deg : 0.0f;
        if (c < din) agg_out[(int64_t)i * din + c] = ac[s];
      }
      if (narrow) {
        const float* wsp[kSlotsIn];   // column clamped into the row: xs / ac are 0 beyond din, so no predicate is needed
        const float* wnp[kSlotsIn];
#pragma unroll
        for (int s = 0; s < kSlotsIn; ++s) {
          const int cc = min(c0 + lane + 32 * s, din - 1);
          wsp[s] = ws + cc * 17;
          wnp[s] = wn + cc * 17;
        }
#pragma unroll
        for (int o = 0; o < 16; ++o) {
          if (o < dout) {      // warp-uniform
            float v = p[o];
#pragma unroll
            for (int s = 0; s < kSlotsIn; ++s) v = fmaf(xs[s], wsp[s][o], fmaf(ac[s], wnp[s][o], v));
            p[o] = v;
          }
        }
      }
    }
    if (narrow) {
      // 16 partial sums per lane, reduced across the warp by a halving butterfly: 8+4+2+1+1
      // shuffles instead of 16 x 5 (the per-output warp_sum made this kernel shuffle-bound)
      bfly<8, 16>(p, lane);
      bfly<4, 8>(p, lane);
      bfly<2, 4>(p, lane);
      bfly<1, 2>(p, lane);
      p[0] += __shfl_xor_sync(0xffffffffu, p[0], 1);
      const int o = ((lane >> 4) & 1) * 8 + ((lane >> 3) & 1) * 4 + ((lane >> 2) & 1) * 2 + ((lane >> 1) & 1);
      if ((lane & 1) == 0 && o < dout) {
        const float v = p[0] + sb[o];
        h_out[(int64_t)i * dout + o] = RELU ? fmaxf(v, 0.0f) : v;
      }
    } else {
      // wider outputs: din <= 128 (one slab, checked at create), xs / ac hold the whole row
      float keep[kSlotsOut] = {0.0f, 0.0f};
      for (int o = 0; o < dout; ++o) {
        float q = 0.0f;
#pragma unroll
        for (int s = 0; s < kSlotsIn; ++s) {
          const int c = lane + 32 * s;
          if (c < din) q += xs[s] * ws[o * din + c] + ac[s] * wn[o * din + c];
        }
        q = warp_sum(q);
        if (lane == (o & 31)) keep[o >> 5] = q + sb[o];
      }
#pragma unroll
      for (int t = 0; t < kSlotsOut; ++t) {
        const int o = lane + 32 * t;
        if (o < dout) h_out[(int64_t)i * dout + o] = RELU ? fmaxf(keep[t], 0.0f) : keep[t];
      }
    }
  }
}

// logits [n][C] -> d_logits in place (softmax - onehot) / n, loss_i[n]
__global__ void __launch_bounds__(128)
k_sage_loss(float* __restrict__ logits, const int32_t* __restrict__ labels, int n, int C,
            float* __restrict__ loss_i) {
  const int i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= n) return;
  float* row = logits + (int64_t)i * C;
  float m = row[0];
  for (int c = 1; c < C; ++c) m = fmaxf(m, row[c]);
  float sum = 0.0f;
  for (int c = 0; c < C; ++c) sum += expf(row[c] - m);
  const float lse = logf(sum);
  const int y = labels[i];
  loss_i[i] = -(row[y] - m - lse);
  const float inv_n = 1.0f / (float)n;
  for (int c = 0; c < C; ++c) {
    const float p = expf(row[c] - m - lse);
    row[c] = (p - (c == y ? 1.0f : 0.0f)) * inv_n;
  }
}

// deterministic mean of loss_i[n] (one CTA, fixed tree)
__global__ void __launch_bounds__(1024) k_sage_loss_mean(const float* __restrict__ loss_i, int n, float* __restrict__ out) {
  __shared__ double sm[1024];
  double acc = 0.0;
  for (int i = threadIdx.x; i < n; i += 1024) acc += (double)loss_i[i];
  sm[threadIdx.x] = acc;
  __syncthreads();
  for (int o = 512; o; o >>= 1) {
    if ((int)threadIdx.x < o) sm[threadIdx.x] += sm[threadIdx.x + o];
    __syncthreads();
  }
  if (threadIdx.x == 0) *out = (float)(sm[0] / (double)n);
}

// d_out [n_dst][dout]: gradient of the loss wrt the layer's activated output.  Accumulates the
// parameter gradients; when d_in != nullptr also the gradient wrt the layer's input rows.
template <bool RELU, bool PARAMS>
__global__ void __launch_bounds__(kSageWarps * 32)
k_sage_bwd(const float* __restrict__ h_in, const float* __restrict__ agg, const float* __restrict__ h_out,
           const float* __restrict__ d_out, const int32_t* __restrict__ indptr,
           const int32_t* __restrict__ src_local, int n_dst, int din, int dout,
           const float* __restrict__ w_self, const float* __restrict__ w_neigh,
           float* __restrict__ g_self, float* __restrict__ g_neigh, float* __restrict__ g_bias,
           float* __restrict__ d_in) {
  extern __shared__ float s_w[];   // [2][dout][din] gradient accumulators (transposed), [dout] bias grads, [2][dout][din] transposed weights
  float* as = s_w;
  float* an = as + din * dout;
  float* ab = an + din * dout;
  float* ws = ab + dout;
  float* wn = ws + dout * din;
  for (int k = threadIdx.x; k < 2 * din * dout + dout; k += blockDim.x) s_w[k] = 0.0f;
  if (d_in) {
    for (int k = threadIdx.x; k < din * dout; k += blockDim.x) {
      const int c = k / dout, o = k - c * dout;
      ws[o * din + c] = w_self[k];
      wn[o * din + c] = w_neigh[k];
    }
  }
  __syncthreads();
  const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
  for (int i = blockIdx.x * kSageWarps + wid; i < n_dst; i += gridDim.x * kSageWarps) {
    float g[kSlotsOut];
#pragma unroll
    for (int t = 0; t < kSlotsOut; ++t) {
      const int o = lane + 32 * t;
      float v = 0.0f;
      if (o < dout) {
        v = d_out[(int64_t)i * dout + o];
        if (RELU && !(h_out[(int64_t)i * dout + o] > 0.0f)) v = 0.0f;
        if (PARAMS && v != 0.0f) atomicAdd(&ab[o], v);
      }
      g[t] = v;
    }
    float xs[kSlotsIn], ag[kSlotsIn], ds[kSlotsIn], da[kSlotsIn];
#pragma unroll
    for (int s = 0; s < kSlotsIn; ++s) {
      const int c = lane + 32 * s;
      xs[s] = c < din ? h_in[(int64_t)i * din + c] : 0.0f;
      ag[s] = c < din ? agg[(int64_t)i * din + c] : 0.0f;
      ds[s] = 0.0f;
      da[s] = 0.0f;
    }
    for (int o = 0; o < dout; ++o) {
      const float go = __shfl_sync(0xffffffffu, g[o >> 5], o & 31);
      if (go == 0.0f) continue;   // warp-uniform
#pragma unroll
      for (int s = 0; s < kSlotsIn; ++s) {
        const int c = lane + 32 * s;
        if (c < din) {
          if (PARAMS) {
            atomicAdd(&as[o * din + c], xs[s] * go);   // transposed: lane-consecutive columns, no bank conflicts
            atomicAdd(&an[o * din + c], ag[s] * go);
          }
          if (d_in) {
            ds[s] += go * ws[o * din + c];
            da[s] += go * wn[o * din + c];
          }
        }
      }
    }
    if (d_in) {
      const int e0 = indptr[i], e1 = indptr[i + 1];
      const float inv = e1 > e0 ? 1.0f / (float)(e1 - e0) : 0.0f;
#pragma unroll
      for (int s = 0; s < kSlotsIn; ++s) {
        const int c = lane + 32 * s;
        if (c < din) atomicAdd(&d_in[(int64_t)i * din + c], ds[s]);
      }
      for (int e = e0; e < e1; ++e) {
        const int64_t src = __ldg(src_local + e);
#pragma unroll
        for (int s = 0; s < kSlotsIn; ++s) {
          const int c = lane + 32 * s;
          if (c < din) atomicAdd(&d_in[src * din + c], da[s] * inv);
        }
      }
    }
  }
  if (!PARAMS) return;
  __syncthreads();
  for (int k = threadIdx.x; k < din * dout; k += blockDim.x) {
    const int c = k / dout, o = k - c * dout;
    const float vs = as[o * din + c], vn = an[o * din + c];
    if (vs != 0.0f) atomicAdd(&g_self[k], vs);
    if (vn != 0.0f) atomicAdd(&g_neigh[k], vn);
  }
  for (int k = threadIdx.x; k < dout; k += blockDim.x)
    if (ab[k] != 0.0f) atomicAdd(&g_bias[k], ab[k]);
}

// Parameter gradients of a layer as a skinny reduction over the destination rows:
//   dW_self = h_in[:n_dst]^T g, dW_neigh = agg^T g, db = sum g,   g = d_out masked by the ReLU.
// Thread t owns input column c = t % 128 and the output half t / 128 (OH outputs) in registers; a CTA
// walks tiles of 64 rows whose g rows sit in shared memory, reading h_in / agg coalesced once.
constexpr int kWgRows = 64;
template <bool RELU, int OH>
__global__ void __launch_bounds__(256)
k_sage_wgrad(const float* __restrict__ h_in, const float* __restrict__ agg, const float* __restrict__ h_out,
             const float* __restrict__ d_out, int n_dst, int din, int dout, int tile_rows,
             float* __restrict__ part /* [gridDim.x][2*din*dout + dout] per-CTA partial sums */) {
  __shared__ float sg[kWgRows][2 * OH];
  const int c = (threadIdx.x & 127) + 128 * blockIdx.y, half = threadIdx.x >> 7;   // blockIdx.y: slab of 128 input columns
  float a_s[OH], a_n[OH];
#pragma unroll
  for (int k = 0; k < OH; ++k) a_s[k] = a_n[k] = 0.0f;
  float a_b = 0.0f;
  const int tiles = (n_dst + tile_rows - 1) / tile_rows;
  for (int t = blockIdx.x; t < tiles; t += gridDim.x) {
    const int r0 = t * tile_rows, rows = min(tile_rows, n_dst - r0);
    __syncthreads();
    for (int k = threadIdx.x; k < tile_rows * 2 * OH; k += 256) {
      const int r = k / (2 * OH), o = k - r * (2 * OH);
      float v = 0.0f;
      if (r < rows && o < dout) {
        v = d_out[(int64_t)(r0 + r) * dout + o];
        if (RELU && !(h_out[(int64_t)(r0 + r) * dout + o] > 0.0f)) v = 0.0f;
      }
      sg[r][o] = v;
    }
    __syncthreads();
    if ((int)threadIdx.x < 2 * OH && blockIdx.y == 0)
      for (int r = 0; r < rows; ++r) a_b += sg[r][threadIdx.x];
    if (c < din) {
#pragma unroll 4
      for (int r = 0; r < rows; ++r) {
        const float xv = __ldg(h_in + (int64_t)(r0 + r) * din + c), av = __ldg(agg + (int64_t)(r0 + r) * din + c);
#pragma unroll
        for (int k = 0; k < OH; ++k) {
          const float gv = sg[r][half * OH + k];
          a_s[k] += xv * gv;
          a_n[k] += av * gv;
        }
      }
    }
  }
  float* mine = part + (int64_t)blockIdx.x * (2 * din * dout + dout);
  if (c < din) {
#pragma unroll
    for (int k = 0; k < OH; ++k) {
      const int o = half * OH + k;
      if (o < dout) {
        mine[c * dout + o] = a_s[k];
        mine[din * dout + c * dout + o] = a_n[k];
      }
    }
  }
  if ((int)threadIdx.x < 2 * OH && (int)threadIdx.x < dout && blockIdx.y == 0) mine[2 * din * dout + threadIdx.x] = a_b;
}

// grads[k] += sum over the CTAs' partials in a fixed order (8 interleaved slices, then the slices
// in order): no atomics, the same bits every run
__global__ void __launch_bounds__(256) k_sage_wreduce(const float* __restrict__ part, int n_part, int P,
                                                      float* __restrict__ grads) {
  __shared__ float sm[8][32];
  const int kx = threadIdx.x & 31, sl = threadIdx.x >> 5;
  const int k = blockIdx.x * 32 + kx;
  float acc = 0.0f;
  if (k < P)
    for (int b = sl; b < n_part; b += 8) acc += part[(int64_t)b * P + k];
  sm[sl][kx] = acc;
  __syncthreads();
  if (sl == 0 && k < P) {
    float t = 0.0f;
#pragma unroll
    for (int q = 0; q < 8; ++q) t += sm[q][kx];
    grads[k] += t;
  }
}

constexpr int kWgMaxGrid = 1024;   // cap on the wgrad grid (sizes the per-CTA partial-sum buffer); the launch takes 4 CTAs per SM
template <bool RELU>
static void launch_wgrad(cudaStream_t st, const float* h_in, const float* agg, const float* h_out, const float* d_out,
                         int n_dst, int din, int dout, float* part, float* grads_layer) {
  // few rows: smaller tiles so that every SM gets one (the tile loop is sequential per CTA)
  int tile_rows = kWgRows;
  while (tile_rows > 8 && (n_dst + tile_rows - 1) / tile_rows < sm_count() * 2) tile_rows >>= 1;
  int grid = (n_dst + tile_rows - 1) / tile_rows;
  const int gmax = std::min(kWgMaxGrid, sm_count() * 4);
  grid = grid < 1 ? 1 : (grid > gmax ? gmax : grid);
  const dim3 g2(grid, (din + 127) / 128);
  if (dout <= 16) k_sage_wgrad<RELU, 8><<<g2, 256, 0, st>>>(h_in, agg, h_out, d_out, n_dst, din, dout, tile_rows, part);
  else if (dout <= 48) k_sage_wgrad<RELU, 24><<<g2, 256, 0, st>>>(h_in, agg, h_out, d_out, n_dst, din, dout, tile_rows, part);
  else k_sage_wgrad<RELU, 32><<<g2, 256, 0, st>>>(h_in, agg, h_out, d_out, n_dst, din, dout, tile_rows, part);
  const int P = 2 * din * dout + dout;
  k_sage_wreduce<<<(P + 31) / 32, 256, 0, st>>>(part, grid, P, grads_layer);
}

__global__ void __launch_bounds__(256) k_sage_sgd(float* __restrict__ p, float* __restrict__ g, int n, float lr) {
  const int i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i < n) {
    p[i] -= lr * g[i];
    g[i] = 0.0f;
  }
}

struct FBuf {
  float* p = nullptr;
  int64_t n = 0;
  cudaError_t ensure(int64_t want, bool* grew) {
    if (want <= n) return cudaSuccess;
    cudaDeviceSynchronize();
    if (p) cudaFree(p);
    p = nullptr;
    n = 0;
    const int64_t cap = want + want / 4 + 1024;
    cudaError_t e = cudaMalloc((void**)&p, (size_t)cap * sizeof(float));
    if (e == cudaSuccess) { n = cap; *grew = true; }
    return e;
  }
};

}  // namespace gg

struct gg_sage {
  int L = 0;
  int dims[GG_MAX_LAYERS + 1] = {0};
  float* params = nullptr;   // per layer: w_self, w_neigh, bias (contiguous)
  float* grads = nullptr;    // same layout
  int64_t off[GG_MAX_LAYERS + 1] = {0};
  int64_t n_params = 0;
  gg::FBuf agg[GG_MAX_LAYERS], out[GG_MAX_LAYERS], dh[GG_MAX_LAYERS], loss_i, part;
  float* loss_dev = nullptr;
};

namespace gg {
static float* p_self(gg_sage* m, int l, float* base) { return base + m->off[l]; }
static float* p_neigh(gg_sage* m, int l, float* base) { return base + m->off[l] + (int64_t)m->dims[l] * m->dims[l + 1]; }
static float* p_bias(gg_sage* m, int l, float* base) { return base + m->off[l] + 2ll * m->dims[l] * m->dims[l + 1]; }
}  // namespace gg

using namespace gg;

extern "C" {

gg_status gg_sage_destroy(gg_sage* m) {
  if (!m) return report_error(GG_ERR_INVALID_ARG, "null model");
  cudaDeviceSynchronize();
  if (m->params) cudaFree(m->params);
  if (m->grads) cudaFree(m->grads);
  if (m->loss_dev) cudaFree(m->loss_dev);
  for (int l = 0; l < GG_MAX_LAYERS; ++l) {
    if (m->agg[l].p) cudaFree(m->agg[l].p);
    if (m->out[l].p) cudaFree(m->out[l].p);
    if (m->dh[l].p) cudaFree(m->dh[l].p);
  }
  if (m->loss_i.p) cudaFree(m->loss_i.p);
  if (m->part.p) cudaFree(m->part.p);
  delete m;
  return GG_OK;
}

gg_status gg_sage_create(int32_t L, const int32_t* dims, const float* const* w_self, const float* const* w_neigh,
                         const float* const* bias, gg_sage** out) {
  if (!dims || !w_self || !w_neigh || !bias || !out) return report_error(GG_ERR_INVALID_ARG, "null argument");
  *out = nullptr;
  if (L < 1 || L > GG_MAX_LAYERS) return report_error(GG_ERR_INVALID_ARG, "num_layers out of range");
  for (int l = 0; l < L; ++l) {
    if (dims[l] < 1 || dims[l + 1] < 1 || dims[l + 1] > 32 * kSlotsOut)
      return report_error(GG_ERR_INVALID_ARG, "dims: outputs must be in [1,64]");
    // a layer's input is walked in slabs of 128 columns when its output is at most 16 wide (the
    // paper's 16 hidden units); only the first layer (the feature tensor) may be wider than 128
    const int max_in = (l == 0 && dims[1] <= 16) ? kSageMaxFeatureDim : 32 * kSlotsIn;
    if (dims[l] > max_in)
      return report_error(GG_ERR_INVALID_ARG, "dims: layer inputs must be in [1,128] (the feature dim up to 1024 when dims[1] <= 16)");
  }
  gg_sage* m = new gg_sage();
  m->L = L;
  for (int l = 0; l <= L; ++l) m->dims[l] = dims[l];
  for (int l = 0; l < L; ++l) m->off[l + 1] = m->off[l] + 2ll * dims[l] * dims[l + 1] + dims[l + 1];
  m->n_params = m->off[L];
  if (cudaMalloc((void**)&m->params, (size_t)m->n_params * sizeof(float)) != cudaSuccess ||
      cudaMalloc((void**)&m->grads, (size_t)m->n_params * sizeof(float)) != cudaSuccess ||
      cudaMalloc((void**)&m->loss_dev, sizeof(float)) != cudaSuccess) {
    cudaGetLastError();
    gg_sage_destroy(m);
    return report_error(GG_ERR_OOM, "device allocation of the model failed");
  }
  cudaMemset(m->grads, 0, (size_t)m->n_params * sizeof(float));
  for (int l = 0; l < L; ++l) {
    const size_t nw = (size_t)dims[l] * dims[l + 1] * sizeof(float);
    cudaMemcpy(p_self(m, l, m->params), w_self[l], nw, cudaMemcpyHostToDevice);
    cudaMemcpy(p_neigh(m, l, m->params), w_neigh[l], nw, cudaMemcpyHostToDevice);
    cudaMemcpy(p_bias(m, l, m->params), bias[l], (size_t)dims[l + 1] * sizeof(float), cudaMemcpyHostToDevice);
  }
  if (cudaDeviceSynchronize() != cudaSuccess) {
    gg_sage_destroy(m);
    return report_error(GG_ERR_CUDA, "copying the initial parameters failed");
  }
  *out = m;
  return GG_OK;
}

gg_status gg_sage_params(gg_sage* m, int32_t l, float* w_self, float* w_neigh, float* bias) {
  if (!m || !w_self || !w_neigh || !bias) return report_error(GG_ERR_INVALID_ARG, "null argument");
  if (l < 0 || l >= m->L) return report_error(GG_ERR_INVALID_ARG, "layer out of range");
  if (cudaDeviceSynchronize() != cudaSuccess) return report_error(GG_ERR_CUDA, "device error before reading parameters");
  const size_t nw = (size_t)m->dims[l] * m->dims[l + 1] * sizeof(float);
  cudaMemcpy(w_self, p_self(m, l, m->params), nw, cudaMemcpyDeviceToHost);
  cudaMemcpy(w_neigh, p_neigh(m, l, m->params), nw, cudaMemcpyDeviceToHost);
  cudaMemcpy(bias, p_bias(m, l, m->params), (size_t)m->dims[l + 1] * sizeof(float), cudaMemcpyDeviceToHost);
  return GG_OK;
}

gg_status gg_sage_step(gg_sage* m, const gg_batch_out* batch, const int32_t* labels, float lr, void* cuda_stream,
                       float* loss_out) {
  if (!m || !batch || !labels || !batch->features) return report_error(GG_ERR_INVALID_ARG, "null argument");
  if (batch->num_layers != m->L) return report_error(GG_ERR_INVALID_ARG, "the batch has a different number of blocks than the model has layers");
  cudaStream_t st = (cudaStream_t)cuda_stream;
  const int L = m->L;
  bool grew = false;
  for (int l = 0; l < L; ++l) {
    const gg_block& b = batch->blocks[L - 1 - l];
    if (m->agg[l].ensure((int64_t)b.n_dst * m->dims[l], &grew) != cudaSuccess ||
        m->out[l].ensure((int64_t)b.n_dst * m->dims[l + 1], &grew) != cudaSuccess ||
        (l > 0 && m->dh[l].ensure((int64_t)b.n_src * m->dims[l], &grew) != cudaSuccess)) {
      cudaGetLastError();
      return report_error(GG_ERR_OOM, "device allocation of the consumer's activations failed");
    }
  }
  const int n_seed = batch->blocks[0].n_dst, C = m->dims[L];
  int64_t max_p = 0;
  for (int l = 0; l < L; ++l) max_p = std::max<int64_t>(max_p, 2ll * m->dims[l] * m->dims[l + 1] + m->dims[l + 1]);
  if (m->loss_i.ensure(n_seed, &grew) != cudaSuccess || m->part.ensure(max_p * kWgMaxGrid, &grew) != cudaSuccess) {
    cudaGetLastError();
    return report_error(GG_ERR_OOM, "device allocation failed");
  }
  static bool attr_set = false;
  if (!attr_set) {
    const int big = 160 * 1024;
    cudaFuncSetAttribute(k_sage_fwd<true>, cudaFuncAttributeMaxDynamicSharedMemorySize, big);
    cudaFuncSetAttribute(k_sage_fwd<false>, cudaFuncAttributeMaxDynamicSharedMemorySize, big);
    cudaFuncSetAttribute(k_sage_bwd<true, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, big);
    cudaFuncSetAttribute(k_sage_bwd<false, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, big);
    attr_set = true;
  }
  const int gcap = sm_count() * 8;
  auto grid_for = [gcap](int n) { int g = (n + kSageWarps - 1) / kSageWarps; return g < 1 ? 1 : (g > gcap ? gcap : g); };
  // forward
  const float* h = (const float*)batch->features;
  for (int l = 0; l < L; ++l) {
    const gg_block& b = batch->blocks[L - 1 - l];
    const int din = m->dims[l], dout = m->dims[l + 1];
    const size_t smem = (size_t)(2 * (dout <= 16 ? 17 * din : din * dout) + dout) * sizeof(float);
    // wide feature rows: the weights take 82 KB per CTA at 602 columns (two CTAs per SM), so each CTA
    // brings 16 warps instead of 8 to keep the row loads of 32 warps per SM in flight
    const int nw = smem > 48 * 1024 ? 2 * kSageWarps : kSageWarps;
    int gf = (b.n_dst + nw - 1) / nw;
    gf = gf < 1 ? 1 : (gf > gcap ? gcap : gf);
    if (l < L - 1)
      k_sage_fwd<true><<<gf, nw * 32, smem, st>>>(h, b.indptr, b.src_local, b.n_dst, din, dout,
          p_self(m, l, m->params), p_neigh(m, l, m->params), p_bias(m, l, m->params), m->agg[l].p, m->out[l].p);
    else
      k_sage_fwd<false><<<gf, nw * 32, smem, st>>>(h, b.indptr, b.src_local, b.n_dst, din, dout,
          p_self(m, l, m->params), p_neigh(m, l, m->params), p_bias(m, l, m->params), m->agg[l].p, m->out[l].p);
    h = m->out[l].p;
  }
  // loss and its gradient (in place in the logits)
  k_sage_loss<<<(n_seed + 127) / 128, 128, 0, st>>>(m->out[L - 1].p, labels, n_seed, C, m->loss_i.p);
  k_sage_loss_mean<<<1, 1024, 0, st>>>(m->loss_i.p, n_seed, loss_out ? loss_out : m->loss_dev);
  // backward
  const float* d_out = m->out[L - 1].p;
  for (int l = L - 1; l >= 0; --l) {
    const gg_block& b = batch->blocks[L - 1 - l];
    const int din = m->dims[l], dout = m->dims[l + 1];
    const float* h_in = l == 0 ? (const float*)batch->features : m->out[l - 1].p;
    float* d_in = l > 0 ? m->dh[l].p : nullptr;
    if (d_in) cudaMemsetAsync(d_in, 0, (size_t)b.n_src * din * sizeof(float), st);
    const size_t smem = (size_t)(4 * din * dout + dout) * sizeof(float);
    if (l < L - 1)
      launch_wgrad<true>(st, h_in, m->agg[l].p, m->out[l].p, d_out, b.n_dst, din, dout, m->part.p, p_self(m, l, m->grads));
    else
      launch_wgrad<false>(st, h_in, m->agg[l].p, m->out[l].p, d_out, b.n_dst, din, dout, m->part.p, p_self(m, l, m->grads));
    if (d_in) {
      if (l < L - 1)
        k_sage_bwd<true, false><<<grid_for(b.n_dst), kSageWarps * 32, smem, st>>>(h_in, m->agg[l].p, m->out[l].p, d_out, b.indptr,
            b.src_local, b.n_dst, din, dout, p_self(m, l, m->params), p_neigh(m, l, m->params),
            p_self(m, l, m->grads), p_neigh(m, l, m->grads), p_bias(m, l, m->grads), d_in);
      else
        k_sage_bwd<false, false><<<grid_for(b.n_dst), kSageWarps * 32, smem, st>>>(h_in, m->agg[l].p, m->out[l].p, d_out, b.indptr,
            b.src_local, b.n_dst, din, dout, p_self(m, l, m->params), p_neigh(m, l, m->params),
            p_self(m, l, m->grads), p_neigh(m, l, m->grads), p_bias(m, l, m->grads), d_in);
    }
    d_out = d_in;
  }
  k_sage_sgd<<<(int)((m->n_params + 255) / 256), 256, 0, st>>>(m->params, m->grads, (int)m->n_params, lr);
  count_launches(4 * L + 2);
  if (cudaGetLastError() != cudaSuccess) return report_error(GG_ERR_CUDA, "a consumer kernel failed to launch");
  return GG_OK;
}

}  // extern "C"
