// NEXT-1: the paper's trace simulator and analytical energy model
// (Eqs. 1-3) on the device.
//
// The trace T = {(b,u) : u in N_b} of one epoch is sampled ONCE by the a-1/a-2
// kernels and kept in HBM (the "Presampled DB" of Fig. 3, here `db_nodes` + `db_off`); sampling
// does not depend on W (reading S7).  For every candidate W the replay below makes a single pass
// over it with the kernels of a-3..a-5 (window unique+count, hot-set select, rebuild delta
// against the previous cache state) plus two small kernels of its own:
//   k_count_db   bumps the packed 8-bit access counters from a window's N_b lists
//   k_classify   per batch: local / cached / miss-per-owner counts (Alg. 1 l.11-12 without
//                moving a byte of features)
// and one more, k_sim_events, which walks the events in trace order (windows ascending, batches
// ascending, owners ascending) and accumulates Eq. 1, Eq. 2 and the stall time of Eq. 3 in IEEE
// double, one rounding per operation (__dadd_rn / __dmul_rn / __ddiv_rn: no FMA contraction), so
// the result is the same bits a CPU gets from the same formulas.
#include "common.cuh"
#include "kernels.h"

namespace gg {

__global__ void __launch_bounds__(256)
k_count_db(const int32_t* __restrict__ db_nodes, int64_t begin, int64_t end, uint32_t* __restrict__ cnt8) {
  const int64_t i = begin + (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (i < end) {
    const int32_t u = __ldg(db_nodes + i);
    atomicAdd(cnt8 + (u >> 2), 1u << (8 * (u & 3)));   // result unused -> RED.ADD
  }
}

// counters[b][0] = hit_local, [1] = hit_cache, [2+m] = |M_{b,m}|; grid (tiles, batches of the window)
__global__ void __launch_bounds__(256)
k_classify(const int32_t* __restrict__ db_nodes, const int64_t* __restrict__ db_off, int b0,
           const int32_t* __restrict__ slot_of, OwnerRanges R, int32_t* __restrict__ counters) {
  __shared__ int32_t s_cnt[2 + GG_MAX_PARTS];
  const int b = b0 + blockIdx.y;
  const int64_t lo = db_off[b], n = db_off[b + 1] - lo;
  const int64_t i0 = (int64_t)blockIdx.x * blockDim.x;
  if (i0 >= n) return;
  if (threadIdx.x < 2 + GG_MAX_PARTS) s_cnt[threadIdx.x] = 0;
  __syncthreads();
  const int64_t i = i0 + threadIdx.x;
  int cls = -1;   // 0 local, 1 cached, 2+m miss
  if (i < n) {
    const int32_t u = __ldg(db_nodes + lo + i);
    const int m = owner_of(R, u);
    cls = m == R.local ? 0 : (__ldg(slot_of + u) >= 0 ? 1 : 2 + m);
  }
  const unsigned l = __ballot_sync(0xffffffffu, cls == 0), c = __ballot_sync(0xffffffffu, cls == 1);
  if ((threadIdx.x & 31) == 0) {
    if (l) atomicAdd(&s_cnt[0], __popc(l));
    if (c) atomicAdd(&s_cnt[1], __popc(c));
  }
  if (cls >= 2) atomicAdd(&s_cnt[cls], 1);
  __syncthreads();
  if (threadIdx.x < 2 + R.P && s_cnt[threadIdx.x])
    atomicAdd(counters + (int64_t)b * (2 + GG_MAX_PARTS) + threadIdx.x, s_cnt[threadIdx.x]);
}

struct SimModel {
  double eps_init[GG_MAX_PARTS], eps_pay_a[GG_MAX_PARTS], eps_pay_b[GG_MAX_PARTS];
  double lam_init[GG_MAX_PARTS], lam_pay_a[GG_MAX_PARTS], lam_pay_b[GG_MAX_PARTS];
  double bw, p_idle;
  int64_t row_bytes;
  int32_t P;
};

// one event with x[o] rows from owner o: adds its Eq. 1 / Eq. 2 term to *e, its duration to *t
__device__ __forceinline__ void sim_event(const int32_t* x, const SimModel& M, double* e, double* t,
                                          long long* events, long long* rows_out) {
  double ev = 0.0, slow = 0.0;
  long long rows = 0;
  for (int o = 0; o < M.P; ++o) {
    const int32_t n = x[o];
    if (n > 0) {
      const double dn = (double)n;
      ev = __dadd_rn(ev, __dadd_rn(M.eps_init[o], __dadd_rn(M.eps_pay_a[o], __dmul_rn(M.eps_pay_b[o], dn))));
      const double tt = __dadd_rn(M.lam_init[o], __dadd_rn(M.lam_pay_a[o], __dmul_rn(M.lam_pay_b[o], dn)));
      if (tt > slow) slow = tt;
      rows += n;
      *events += 1;
    }
  }
  *e = __dadd_rn(*e, ev);
  if (rows > 0) {
    const double ceil_t = __ddiv_rn((double)(rows * M.row_bytes), M.bw);
    *t = __dadd_rn(*t, slow > ceil_t ? slow : ceil_t);
  }
  *rows_out += rows;
}

// delta: [K][GG_MAX_PARTS] (|Delta_{k,m}|), counters: [B][2+GG_MAX_PARTS]
__global__ void k_sim_events(const int32_t* __restrict__ delta, const int32_t* __restrict__ counters,
                             int K, int B, int W, SimModel M, gg_sim_result* __restrict__ out) {
  if (blockIdx.x != 0 || threadIdx.x != 0) return;
  double e_rebuild = 0.0, e_miss = 0.0, t_stall = 0.0;
  long long rebuild_events = 0, miss_events = 0, rebuild_rows = 0, miss_rows = 0, hit_local = 0, hit_cache = 0;
  for (int k = 0; k < K; ++k) {
    sim_event(delta + (int64_t)k * GG_MAX_PARTS, M, &e_rebuild, &t_stall, &rebuild_events, &rebuild_rows);
    const int b1 = min(B, (k + 1) * W);
    for (int b = k * W; b < b1; ++b) {
      const int32_t* c = counters + (int64_t)b * (2 + GG_MAX_PARTS);
      hit_local += c[0];
      hit_cache += c[1];
      sim_event(c + 2, M, &e_miss, &t_stall, &miss_events, &miss_rows);
    }
  }
  const double e_stall = __dmul_rn(M.p_idle, t_stall);
  const long long remote = hit_cache + miss_rows;
  out->W = W;
  out->n_windows = K;
  out->rebuild_events = rebuild_events;
  out->miss_events = miss_events;
  out->rebuild_rows = rebuild_rows;
  out->miss_rows = miss_rows;
  out->n_access = hit_local + remote;
  out->n_remote_access = remote;
  out->hit_local = hit_local;
  out->hit_cache = hit_cache;
  out->e_rebuild = e_rebuild;
  out->e_miss = e_miss;
  out->t_stall = t_stall;
  out->e_stall = e_stall;
  out->e_phy = __dadd_rn(__dadd_rn(e_rebuild, e_miss), e_stall);
  out->hit_ratio = remote ? __ddiv_rn((double)hit_cache, (double)remote) : 1.0;
}

// ---- NEXT-3: rank calibration, Eq. (5) of PAPER.md:226-237 ----------------------------------------
// S(W) = beta^T z(W) + gamma_W; L = sum_{i<j} log(1 + exp(-sigma_ij (S_j - S_i))) + lambda ||beta||^2.
// Seven candidates and a handful of features: one thread walks the pairs in a fixed order, so
// the only difference from a CPU run of the same steps is the last ulp of exp().
constexpr int kCalMaxN = 64, kCalMaxF = 16;
__global__ void k_rank_calibrate(const double* __restrict__ Z, const double* __restrict__ e_gt, int n, int F,
                                 double lam, double lr, int iters, double* __restrict__ beta_out,
                                 double* __restrict__ gamma_out, double* __restrict__ loss_out) {
  if (blockIdx.x != 0 || threadIdx.x != 0) return;
  double beta[kCalMaxF], gamma[kCalMaxN], S[kCalMaxN], dS[kCalMaxN];
  for (int f = 0; f < F; ++f) beta[f] = 0.0;
  for (int i = 0; i < n; ++i) gamma[i] = 0.0;
  for (int it = 0; it <= iters; ++it) {
    for (int i = 0; i < n; ++i) {
      double acc = 0.0;
      for (int f = 0; f < F; ++f) acc = __dadd_rn(acc, __dmul_rn(beta[f], Z[i * F + f]));
      S[i] = __dadd_rn(acc, gamma[i]);
      dS[i] = 0.0;
    }
    if (it == iters) break;
    for (int i = 0; i < n; ++i)
      for (int j = i + 1; j < n; ++j) {
        const double d = e_gt[j] - e_gt[i];
        const double sg = d > 0 ? 1.0 : (d < 0 ? -1.0 : 0.0);
        if (sg == 0.0) continue;
        const double g = __ddiv_rn(-sg, __dadd_rn(1.0, exp(__dmul_rn(sg, __dadd_rn(S[j], -S[i])))));
        dS[j] = __dadd_rn(dS[j], g);
        dS[i] = __dadd_rn(dS[i], -g);
      }
    for (int f = 0; f < F; ++f) {
      double acc = 0.0;
      for (int i = 0; i < n; ++i) acc = __dadd_rn(acc, __dmul_rn(dS[i], Z[i * F + f]));
      beta[f] = __dadd_rn(beta[f], -__dmul_rn(lr, __dadd_rn(acc, __dmul_rn(__dmul_rn(2.0, lam), beta[f]))));
    }
    for (int i = 0; i < n; ++i) gamma[i] = __dadd_rn(gamma[i], -__dmul_rn(lr, dS[i]));
  }
  double loss = 0.0;
  for (int i = 0; i < n; ++i)
    for (int j = i + 1; j < n; ++j) {
      const double d = e_gt[j] - e_gt[i];
      const double sg = d > 0 ? 1.0 : (d < 0 ? -1.0 : 0.0);
      loss += log1p(exp(-sg * (S[j] - S[i])));
    }
  double b2 = 0.0;
  for (int f = 0; f < F; ++f) b2 += beta[f] * beta[f];
  *loss_out = loss + lam * b2;
  for (int f = 0; f < F; ++f) beta_out[f] = beta[f];
  for (int i = 0; i < n; ++i) gamma_out[i] = gamma[i];
}

cudaError_t rank_calibrate(const double* z_host, const double* e_host, int n, int F, double lam, double lr,
                           int iters, double* beta_host, double* gamma_host, double* loss_host) {
  if (n < 1 || n > kCalMaxN || F < 0 || F > kCalMaxF) return cudaErrorInvalidValue;
  double* d = nullptr;
  const size_t nz = (size_t)n * (F > 0 ? F : 1);
  cudaError_t e = cudaMalloc((void**)&d, (nz + 2 * n + kCalMaxF + 1) * sizeof(double));
  if (e != cudaSuccess) return e;
  double *dZ = d, *dE = d + nz, *dB = dE + n, *dG = dB + kCalMaxF, *dL = dG + n;
  if (F > 0) cudaMemcpy(dZ, z_host, (size_t)n * F * sizeof(double), cudaMemcpyHostToDevice);
  cudaMemcpy(dE, e_host, (size_t)n * sizeof(double), cudaMemcpyHostToDevice);
  k_rank_calibrate<<<1, 32>>>(dZ, dE, n, F, lam, lr, iters, dB, dG, dL);
  count_launches(1);
  e = cudaDeviceSynchronize();
  if (e == cudaSuccess) {
    if (F > 0) cudaMemcpy(beta_host, dB, (size_t)F * sizeof(double), cudaMemcpyDeviceToHost);
    cudaMemcpy(gamma_host, dG, (size_t)n * sizeof(double), cudaMemcpyDeviceToHost);
    cudaMemcpy(loss_host, dL, sizeof(double), cudaMemcpyDeviceToHost);
    e = cudaGetLastError();
  }
  cudaFree(d);
  return e;
}

void launch_count_db(cudaStream_t st, const int32_t* db_nodes, int64_t begin, int64_t end, uint32_t* cnt8) {
  if (end <= begin) return;
  const int64_t n = end - begin;
  k_count_db<<<(unsigned)((n + 255) / 256), 256, 0, st>>>(db_nodes, begin, end, cnt8);
  count_launches(1);
}

void launch_classify(cudaStream_t st, const int32_t* db_nodes, const int64_t* db_off, int b0, int nb,
                     int64_t max_n, const int32_t* slot_of, const OwnerRanges& R, int32_t* counters) {
  if (nb <= 0 || max_n <= 0) return;
  dim3 grid((unsigned)((max_n + 255) / 256), nb);
  k_classify<<<grid, 256, 0, st>>>(db_nodes, db_off, b0, slot_of, R, counters);
  count_launches(1);
}

void launch_sim_events(cudaStream_t st, const int32_t* delta, const int32_t* counters, int K, int B, int W,
                       const gg_energy_model& E, int P, int64_t row_bytes, gg_sim_result* out_dev) {
  SimModel M;
  for (int o = 0; o < GG_MAX_PARTS; ++o) {
    M.eps_init[o] = E.eps_init[o]; M.eps_pay_a[o] = E.eps_pay_a[o]; M.eps_pay_b[o] = E.eps_pay_b[o];
    M.lam_init[o] = E.lam_init[o]; M.lam_pay_a[o] = E.lam_pay_a[o]; M.lam_pay_b[o] = E.lam_pay_b[o];
  }
  M.bw = E.bw_bytes_per_s; M.p_idle = E.p_idle_w; M.row_bytes = row_bytes; M.P = P;
  k_sim_events<<<1, 32, 0, st>>>(delta, counters, K, B, W, M, out_dev);
  count_launches(1);
}

}  // namespace gg
