// sm_100a kernels of the DMRG hot path and the CUDA backend.
//
// k_gemm_f64: the one generic, output-stationary grouped GEMM that executes every descriptor
// list of plan.cpp (H_eff stage 1 / stage 2, rotation, integral contraction):
//     C[m][n] = colscale[n / n1] * sum_seg alpha_seg * sum_k A_seg[m][k] B_seg[k][n]
// Native FP64 on the tensor pipe: tcgen05 has no FP64 kind on sm_100a (ptxas rejects
// .kind::f64), so the FP64 path is warp-level mma.sync.m8n8k4.f64 (SASS DMMA.8x8x4) fed from
// XOR-swizzled shared-memory tiles (SURVEY.md section 0 "Survey-time hardware facts", 7).
// Each CTA owns one output tile and walks that tile's segment list, accumulating in registers:
// no atomics, deterministic, one write per output element.
#include <cuda_runtime.h>

#include <cstdio>
#include <cstdlib>
#include <algorithm>
#include <map>
#include <new>
#include <queue>
#include <stdexcept>
#include <string>
#include <vector>

#include "backend.h"
#include "gemm_f64.cuh"
#include "tc_i8.cuh"
#include "emu.cuh"
#include "emu_seg.cuh"
#include "emu_s1.cuh"
#include "tf32_seg.cuh"

namespace dmrg {

// 8 independent FP64 FMA chains per thread (measurement only, dmrg_measure_peak(3))
__global__ void __launch_bounds__(256) k_peak_dfma(int iters, double *sink, double a) {
  double x[8];
#pragma unroll
  for (int i = 0; i < 8; ++i) x[i] = 1e-3 * (threadIdx.x + i);
  const double b = a * 1e-9;
  for (int it = 0; it < iters; ++it) {
#pragma unroll
    for (int i = 0; i < 8; ++i) x[i] = fma(x[i], a, b);
  }
  double s = 0;
#pragma unroll
  for (int i = 0; i < 8; ++i) s += x[i];
  if (s == 12345.678) *sink = s;
}

#define CK(call)                                                                          \
  do {                                                                                    \
    cudaError_t e_ = (call);                                                              \
    if (e_ != cudaSuccess)                                                                \
      throw std::runtime_error(std::string("CUDA: ") + cudaGetErrorString(e_) + " at " #call); \
  } while (0)

// a7: diag(H_eff)[l][r] = sum_t f_t diag(O_L,t)[l] diag(O_R,t)[r], one CTA per psi block.  The diagonals of 8 terms
// at a time are gathered into shared memory (they are strided in HBM: stride d + 1) and every thread accumulates its
// elements from there in a fixed order, so each diagonal element is read from global memory once per block.
static constexpr int DIAG_TERMS = 8, DIAG_MAXD = 320;       // 40 KB of static shared memory
__global__ void __launch_bounds__(1024) k_heff_diag(const DiagJob *__restrict__ jobs,
                                                   const DiagTerm *__restrict__ terms, BufTable bufs,
                                                   double *__restrict__ out) {
  const DiagJob j = jobs[blockIdx.x];
  const int nel = j.dL * j.dR;
  if (j.dL > DIAG_MAXD || j.dR > DIAG_MAXD) {          // sectors beyond the staging buffers: straight from global memory
    for (int e = threadIdx.x; e < nel; e += blockDim.x) {
      int l = e / j.dR, r = e - l * j.dR;
      double s = 0.0;
      for (int t = j.t_begin; t < j.t_end; ++t) {
        const DiagTerm dt = terms[t];
        s += dt.f * __ldg(rd_ref(bufs, dt.l) + (int64_t)l * dt.ls) * __ldg(rd_ref(bufs, dt.r) + (int64_t)r * dt.rs);
      }
      out[j.off + e] = s;
    }
    return;
  }
  __shared__ double sl[DIAG_TERMS][DIAG_MAXD], sr[DIAG_TERMS][DIAG_MAXD];
  constexpr int EPT = 16;                              // elements per thread and sweep: one sweep covers 16384 elements
  const int NT = blockDim.x;
  for (int e0 = 0; e0 < nel; e0 += NT * EPT) {
    double acc[EPT];
    int li[EPT], ri[EPT];
#pragma unroll
    for (int q = 0; q < EPT; ++q) {
      const int e = e0 + q * NT + threadIdx.x;
      acc[q] = 0.0;
      li[q] = e < nel ? e / j.dR : 0;
      ri[q] = e < nel ? e - li[q] * j.dR : 0;
    }
    for (int t0 = j.t_begin; t0 < j.t_end; t0 += DIAG_TERMS) {
      const int nt = min(DIAG_TERMS, j.t_end - t0);
      __syncthreads();
      for (int idx = threadIdx.x; idx < nt * (j.dL + j.dR); idx += NT) {
        const int t = idx / (j.dL + j.dR), k = idx - t * (j.dL + j.dR);
        const DiagTerm dt = terms[t0 + t];
        if (k < j.dL) sl[t][k] = dt.f * __ldg(rd_ref(bufs, dt.l) + (int64_t)k * dt.ls);
        else sr[t][k - j.dL] = __ldg(rd_ref(bufs, dt.r) + (int64_t)(k - j.dL) * dt.rs);
      }
      __syncthreads();
      for (int t = 0; t < nt; ++t) {
#pragma unroll
        for (int q = 0; q < EPT; ++q) acc[q] = fma(sl[t][li[q]], sr[t][ri[q]], acc[q]);
      }
    }
#pragma unroll
    for (int q = 0; q < EPT; ++q) {
      const int e = e0 + q * NT + threadIdx.x;
      if (e < nel) out[j.off + e] = acc[q];
    }
  }
}

// Fixed-order sum of the stage-2 K-chunk partials of one psi block (one CTA per block).
__global__ void __launch_bounds__(128) k_reduce_partials(const ReduceJob *__restrict__ jobs,
                                                         const double *__restrict__ partial,
                                                         double *__restrict__ out) {
  const ReduceJob j = jobs[blockIdx.x];
  for (int e = threadIdx.x; e < j.mn; e += blockDim.x) {
    const double *p = partial + j.part + e;
    double s = 0.0;
    for (int c = 0; c < j.n_chunks; ++c) s += p[(int64_t)c * j.mn];
    out[j.out + e] = s;
  }
}

// ------------------------------------------------------------------ Davidson vector kernels (a8)
static constexpr int DOT_BLOCKS = 296, DOT_THREADS = 256, MAX_BASIS = 32;

__global__ void __launch_bounds__(DOT_THREADS) k_dots_partial(const double *__restrict__ V, int64_t ld, int nvec,
                                                              const double *__restrict__ w, int64_t n,
                                                              double *__restrict__ partial) {
  __shared__ double red[DOT_THREADS / 32];
  for (int v = 0; v < nvec; ++v) {
    const double *x = V + (int64_t)v * ld;
    double s = 0.0;
    for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (int64_t)gridDim.x * blockDim.x)
      s += x[i] * w[i];
    for (int o = 16; o > 0; o >>= 1) s += __shfl_xor_sync(0xffffffffu, s, o);
    if ((threadIdx.x & 31) == 0) red[threadIdx.x >> 5] = s;
    __syncthreads();
    if (threadIdx.x == 0) {
      double t = 0.0;
      for (int i = 0; i < DOT_THREADS / 32; ++i) t += red[i];
      partial[(int64_t)v * gridDim.x + blockIdx.x] = t;
    }
    __syncthreads();
  }
}
// Row a4 of the 3xTF32 mode on its own (dmrg_tf32_split): the split the slicing kernels and stage-1 epilogues apply
__global__ void __launch_bounds__(256) k_tf32_split(const double *__restrict__ x, int64_t n, uint32_t *__restrict__ hi,
                                                    uint32_t *__restrict__ lo) {
  for (int64_t i = blockIdx.x * 256ll + threadIdx.x; i < n; i += (int64_t)gridDim.x * 256) tf32_split(x[i], hi[i], lo[i]);
}
__global__ void k_dots_final(const double *__restrict__ partial, int nblocks, double *__restrict__ out) {
  // one warp per vector, fixed summation order
  const double *p = partial + (int64_t)blockIdx.x * nblocks;
  double s = 0.0;
  for (int i = threadIdx.x; i < nblocks; i += 32) s += p[i];
  for (int o = 16; o > 0; o >>= 1) s += __shfl_xor_sync(0xffffffffu, s, o);
  if (threadIdx.x == 0) out[blockIdx.x] = s;
}

// Append column `col` (V^T w) to the Gram matrix G and diagonalise G (m x m, symmetric) with
// cyclic Jacobi in one thread: m <= 64, a few thousand flops.  Writes the lowest eigenpair.
__global__ void k_davidson_small(double *G, int ldg, int m, const double *col, double *y, double *theta_out) {
  __shared__ double A[MAX_BASIS * MAX_BASIS], Vv[MAX_BASIS * MAX_BASIS];
  if (threadIdx.x != 0) return;
  for (int j = 0; j < m; ++j) { G[j * ldg + (m - 1)] = col[j]; G[(m - 1) * ldg + j] = col[j]; }
  for (int i = 0; i < m; ++i)
    for (int j = 0; j < m; ++j) { A[i * m + j] = G[i * ldg + j]; Vv[i * m + j] = (i == j) ? 1.0 : 0.0; }
  for (int sweep = 0; sweep < 40; ++sweep) {
    double off = 0.0, nrm = 0.0;
    for (int i = 0; i < m; ++i)
      for (int j = 0; j < m; ++j) { double a = A[i * m + j]; nrm += a * a; if (i != j) off += a * a; }
    if (off <= 1e-30 * nrm || off == 0.0) break;
    for (int p = 0; p < m - 1; ++p)
      for (int q = p + 1; q < m; ++q) {
        double apq = A[p * m + q];
        if (fabs(apq) <= 1e-300) continue;
        double th = (A[q * m + q] - A[p * m + p]) / (2.0 * apq);
        double t = (th >= 0 ? 1.0 : -1.0) / (fabs(th) + sqrt(th * th + 1.0));
        double c = 1.0 / sqrt(t * t + 1.0), s = t * c;
        for (int k = 0; k < m; ++k) {
          double akp = A[k * m + p], akq = A[k * m + q];
          A[k * m + p] = c * akp - s * akq; A[k * m + q] = s * akp + c * akq;
        }
        for (int k = 0; k < m; ++k) {
          double apk = A[p * m + k], aqk = A[q * m + k];
          A[p * m + k] = c * apk - s * aqk; A[q * m + k] = s * apk + c * aqk;
        }
        for (int k = 0; k < m; ++k) {
          double vkp = Vv[k * m + p], vkq = Vv[k * m + q];
          Vv[k * m + p] = c * vkp - s * vkq; Vv[k * m + q] = s * vkp + c * vkq;
        }
      }
  }
  int best = 0;
  for (int i = 1; i < m; ++i) if (A[i * m + i] < A[best * m + best]) best = i;
  *theta_out = A[best * m + best];
  for (int k = 0; k < m; ++k) y[k] = Vv[k * m + best];
}

// x = V y,  r = W y - theta x
__global__ void k_ritz_residual(const double *__restrict__ V, const double *__restrict__ W, int64_t ld, int m,
                                int64_t n, const double *__restrict__ y, const double *__restrict__ theta,
                                double *__restrict__ x, double *__restrict__ r) {
  __shared__ double ys[MAX_BASIS];
  if (threadIdx.x < m) ys[threadIdx.x] = y[threadIdx.x];
  __syncthreads();
  const double th = *theta;
  for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (int64_t)gridDim.x * blockDim.x) {
    double xv = 0.0, wv = 0.0;
    for (int k = 0; k < m; ++k) { xv += ys[k] * V[(int64_t)k * ld + i]; wv += ys[k] * W[(int64_t)k * ld + i]; }
    x[i] = xv;
    r[i] = wv - th * xv;
  }
}
// t_i = r_i / (theta - diag_i), |theta - diag_i| < 1e-12 replaced by +-1e-12
__global__ void k_precondition(const double *__restrict__ r, const double *__restrict__ diag,
                               const double *__restrict__ theta, double *__restrict__ t, int64_t n) {
  const double th = *theta;
  for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (int64_t)gridDim.x * blockDim.x) {
    double den = th - diag[i];
    if (fabs(den) < 1e-12) den = den < 0 ? -1e-12 : 1e-12;
    t[i] = r[i] / den;
  }
}
// t -= V c
__global__ void k_subtract_projection(const double *__restrict__ V, int64_t ld, int m, const double *__restrict__ c,
                                      double *__restrict__ t, int64_t n) {
  __shared__ double cs[MAX_BASIS];
  if (threadIdx.x < m) cs[threadIdx.x] = c[threadIdx.x];
  __syncthreads();
  for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (int64_t)gridDim.x * blockDim.x) {
    double s = 0.0;
    for (int k = 0; k < m; ++k) s += cs[k] * V[(int64_t)k * ld + i];
    t[i] -= s;
  }
}
__global__ void k_scale_inv_norm(const double *__restrict__ src, const double *__restrict__ nrm2,
                                 double *__restrict__ dst, int64_t n) {
  const double s = 1.0 / sqrt(*nrm2);
  for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (int64_t)gridDim.x * blockDim.x)
    dst[i] = src[i] * s;
}

// Register-resident DMMA loop: the measuring stick for the FP64 tensor-pipe peak (8(d)).
__global__ void __launch_bounds__(256) k_peak_dmma(int iters, double *sink) {
  double acc[16][2];
#pragma unroll
  for (int i = 0; i < 16; ++i) { acc[i][0] = 0.0; acc[i][1] = 0.0; }
  double a = 1.0 + threadIdx.x * 1e-9, b = 1.0 - threadIdx.x * 1e-9;
  for (int it = 0; it < iters; ++it) {
#pragma unroll
    for (int i = 0; i < 16; ++i) dmma884(acc[i][0], acc[i][1], a, b);
  }
  double s = 0.0;
#pragma unroll
  for (int i = 0; i < 16; ++i) s += acc[i][0] + acc[i][1];
  if (s == 123.456) sink[0] = s;
}

// ------------------------------------------------------------------ backend
class CudaBackend : public Backend {
 public:
  int device;
  cudaStream_t stream;
  double *dot_partial = nullptr;
  cudaEvent_t ev[12];
  int n_sm = 148;

  CudaBackend(int dev, void *st) : device(dev), stream((cudaStream_t)st) {
    CK(cudaSetDevice(dev));
    cudaDeviceProp prop;
    CK(cudaGetDeviceProperties(&prop, dev));
    if (prop.major != 10) throw std::runtime_error("this library targets sm_100 (B200) only; found sm_" +
                                                   std::to_string(prop.major) + std::to_string(prop.minor));
    n_sm = prop.multiProcessorCount;
    CK(cudaMalloc(&dot_partial, sizeof(double) * DOT_BLOCKS * MAX_BASIS));
    for (auto &e : ev) CK(cudaEventCreate(&e));
    set_smem<0>(); set_smem<1>(); set_smem<2>(); set_smem<3>(); set_smem<4>();
  }
  template <int ROLE> void set_smem() {
    CK(cudaFuncSetAttribute(k_gemm_f64<3, ROLE>, cudaFuncAttributeMaxDynamicSharedMemorySize, GemmCfg<3>::SMEM_BYTES));
    CK(cudaFuncSetAttribute(k_gemm_f64<4, ROLE>, cudaFuncAttributeMaxDynamicSharedMemorySize, GemmCfg<4>::SMEM_BYTES));
  }
  ~CudaBackend() override {
    cudaFree(dot_partial);
    for (auto &e : ev) cudaEventDestroy(e);
  }
  void make_current() override {
    int cur = -1;
    if (cudaGetDevice(&cur) != cudaSuccess || cur != device) CK(cudaSetDevice(device));
  }
  void *alloc(size_t bytes) override {
    void *p = nullptr;
    if (bytes == 0) bytes = 8;
    cudaError_t e = cudaMalloc(&p, bytes);
    if (e != cudaSuccess) { cudaGetLastError(); throw std::bad_alloc(); }
    return p;
  }
  void release(void *p) override { if (p) cudaFree(p); }
  void upload(void *dst, const void *src, size_t bytes) override {
    if (bytes) CK(cudaMemcpyAsync(dst, src, bytes, cudaMemcpyHostToDevice, stream));
  }
  void download(void *dst, const void *src, size_t bytes) override {
    if (bytes) CK(cudaMemcpyAsync(dst, src, bytes, cudaMemcpyDeviceToHost, stream));
    CK(cudaStreamSynchronize(stream));
  }
  void copy(void *dst, const void *src, size_t bytes) override {
    if (bytes) CK(cudaMemcpyAsync(dst, src, bytes, cudaMemcpyDeviceToDevice, stream));
  }
  void zero(void *dst, size_t bytes) override { if (bytes) CK(cudaMemsetAsync(dst, 0, bytes, stream)); }
  void sync() override { CK(cudaStreamSynchronize(stream)); }

  template <class T> void *up(const std::vector<T> &v) {
    void *p = alloc(sizeof(T) * v.size());
    upload(p, v.data(), sizeof(T) * v.size());
    return p;
  }
  void upload_jobs(const JobList &jl, DevJobList &out, int role) override {
    free_jobs(out);
    out.role = role; out.tile = jl.tile;
    out.n_jobs = (int)jl.jobs.size(); out.n_segs = (int)jl.segs.size(); out.n_tiles = (int)jl.tiles.size();
    out.flops = jl.flops;
    out.jobs = up(jl.jobs); out.segs = up(jl.segs); out.tiles = up(jl.tiles);
    CK(cudaStreamSynchronize(stream));   // the host vectors may die after this call
  }
  void free_jobs(DevJobList &jl) override {
    release(jl.jobs); release(jl.segs); release(jl.tiles);
    jl = DevJobList();
  }
  void upload_diag(const std::vector<DiagJob> &jobs, const std::vector<DiagTerm> &terms, DevDiag &out) override {
    free_diag(out);
    out.n_jobs = (int)jobs.size();
    out.jobs = up(jobs); out.terms = up(terms);
    CK(cudaStreamSynchronize(stream));
  }
  void free_diag(DevDiag &d) override { release(d.jobs); release(d.terms); d = DevDiag(); }
  void upload_reduce(const std::vector<ReduceJob> &jobs, DevReduce &out) override {
    free_reduce(out);
    out.n_jobs = (int)jobs.size();
    out.jobs = up(jobs);
    CK(cudaStreamSynchronize(stream));
  }
  void free_reduce(DevReduce &d) override { release(d.jobs); d = DevReduce(); }
  void run_reduce(const DevReduce &d, const double *partial, double *out) override {
    if (d.n_jobs == 0) return;
    ++n_launches;
    k_reduce_partials<<<d.n_jobs, 128, 0, stream>>>((const ReduceJob *)d.jobs, partial, out);
    CK(cudaGetLastError());
  }

  void run_jobs(const DevJobList &jl, const BufTable &bufs) override {
    if (jl.n_tiles == 0) return;
    const JobDesc *j = (const JobDesc *)jl.jobs;
    const SegDesc *sg = (const SegDesc *)jl.segs;
    const TileDesc *t = (const TileDesc *)jl.tiles;
#define LAUNCH(MT, ROLE) \
    (++n_launches, k_gemm_f64<MT, ROLE><<<jl.n_tiles, 128, GemmCfg<MT>::SMEM_BYTES, stream>>>(j, sg, t, bufs))
#define LAUNCH_ROLE(MT)                                                   \
    switch (jl.role) {                                                    \
      case 0: LAUNCH(MT, 0); break; case 1: LAUNCH(MT, 1); break;         \
      case 2: LAUNCH(MT, 2); break; case 3: LAUNCH(MT, 3); break;         \
      default: LAUNCH(MT, 4); break;                                      \
    }
    switch (jl.tile) {
      case 32: LAUNCH_ROLE(2); break;
      case 48: LAUNCH_ROLE(3); break;
      case 64: LAUNCH_ROLE(4); break;
      default: throw std::runtime_error("unsupported tile size");
    }
#undef LAUNCH_ROLE
#undef LAUNCH
    CK(cudaGetLastError());
  }
  void run_diag(const DevDiag &d, const BufTable &bufs, double *out) override {
    if (d.n_jobs == 0) return;
    ++n_launches;
    k_heff_diag<<<d.n_jobs, 1024, 0, stream>>>((const DiagJob *)d.jobs, (const DiagTerm *)d.terms, bufs, out);
    CK(cudaGetLastError());
  }
  int vec_blocks(int64_t n) const { return (int)std::max<int64_t>(1, std::min<int64_t>((n + 255) / 256, 4 * n_sm)); }
  void dots(const double *V, int64_t ld, int nvec, const double *w, int64_t n, double *out) override {
    if (nvec > MAX_BASIS) throw std::runtime_error("too many basis vectors");
    ++n_launches;
    k_dots_partial<<<DOT_BLOCKS, DOT_THREADS, 0, stream>>>(V, ld, nvec, w, n, dot_partial);
    ++n_launches;
    k_dots_final<<<nvec, 32, 0, stream>>>(dot_partial, DOT_BLOCKS, out);
    CK(cudaGetLastError());
  }
  void davidson_small(double *G, int ldg, int m, const double *col, double *y, double *theta_out) override {
    if (m > MAX_BASIS) throw std::runtime_error("Davidson basis too large");
    ++n_launches;
    k_davidson_small<<<1, 32, 0, stream>>>(G, ldg, m, col, y, theta_out);
    CK(cudaGetLastError());
  }
  void ritz_residual(const double *V, const double *W, int64_t ld, int m, int64_t n, const double *y,
                     const double *theta, double *x, double *r) override {
    ++n_launches;
    k_ritz_residual<<<vec_blocks(n), 256, 0, stream>>>(V, W, ld, m, n, y, theta, x, r);
    CK(cudaGetLastError());
  }
  void precondition(const double *r, const double *diag, const double *theta, double *t, int64_t n) override {
    ++n_launches;
    k_precondition<<<vec_blocks(n), 256, 0, stream>>>(r, diag, theta, t, n);
    CK(cudaGetLastError());
  }
  void subtract_projection(const double *V, int64_t ld, int m, const double *c, double *t, int64_t n) override {
    ++n_launches;
    k_subtract_projection<<<vec_blocks(n), 256, 0, stream>>>(V, ld, m, c, t, n);
    CK(cudaGetLastError());
  }
  void scale_inv_norm(const double *src, const double *nrm2, double *dst, int64_t n) override {
    ++n_launches;
    k_scale_inv_norm<<<vec_blocks(n), 256, 0, stream>>>(src, nrm2, dst, n);
    CK(cudaGetLastError());
  }
  void tf32_split_run(const double *src, int64_t n, uint32_t *hi, uint32_t *lo) override {
    if (n < 1) return;
    ++n_launches;
    k_tf32_split<<<vec_blocks(n), 256, 0, stream>>>(src, n, hi, lo);
    CK(cudaGetLastError());
  }
  void emu_slice(const double *src, int lines, int K, int64_t ls, int64_t ks, int kappa, signed char *out,
                 int *expo) override {
    if (kappa < 2 || kappa > EMU_MAX_KAPPA) throw std::invalid_argument("slices must be in [2, 7]");
    ++n_launches;
    k_emu_slice<<<lines, 128, 0, stream>>>(src, lines, K, ls, ks, kappa, (int8_t *)out, lines, K, expo, K);
    CK(cudaGetLastError());
  }
  // C = A B through the same descriptors as stage 2: one segment per K chunk of at most 16384 (kappa products
  // of magnitude 2^14 summed over the chunk stay below 2^31, Appendix A6 step 4), exponents per chunk.
  void emu_gemm(int M, int N, int K, const double *A, const double *B, double *C, int kappa, int keep, double *ms_slice,
                double *ms_gemm) override {
    if (kappa < 2 || kappa > EMU_MAX_KAPPA) throw std::invalid_argument("slices must be in [2, 7]");
    if (keep < 1 || keep > kappa) throw std::invalid_argument("emu_gemm: keep must be in [1, slices]");
    if (M < 1 || N < 1 || K < 1) throw std::invalid_argument("emu_gemm: empty problem");
    const int kchunk = 16384, n_chunks = (K + kchunk - 1) / kchunk;
    HeffPlan P;                                  // only the emulated lists are used
    P.emu.assign(1, EmuPass());
    EmuPass &E = P.emu[0];
    EmuJob job{};
    job.c = mkref(B_NEW, 0); job.scale = -1; job.n1 = FLAT; job.M = M; job.N = N; job.c_ld = N; job.seg_begin = 0; job.seg_end = n_chunks;
    for (int c = 0; c < n_chunks; ++c) {
      const int k0 = c * kchunk, kc = std::min(kchunk, K - k0), kpad = (kc + 31) / 32 * 32;
      EmuSliceDesc da{}, db{};
      da.src = mkref(B_OPS_L, k0); da.mstride = 0; da.lstride = 1; da.linestride = K;            // rows of A
      da.n_members = 1; da.dl = da.dlpad = kc; da.lines = M; da.ld = kpad; da.tile_rows = EMU_BM;
      da.out_off = P.emuL_bytes; da.exp_off = P.expL_n;
      P.emuL_bytes += (int64_t)(M + EMU_BM - 1) / EMU_BM * EMU_BM * kpad; P.expL_n += M;
      db.src = mkref(B_OPS_R, (int64_t)k0 * N); db.mstride = 0; db.lstride = N; db.linestride = 1;   // columns of B
      db.n_members = 1; db.dl = db.dlpad = kc; db.lines = N; db.ld = kpad; db.tile_rows = EMU_BN;
      db.out_off = P.emuT_bytes; db.exp_off = P.expT_n;
      P.emuT_bytes += (int64_t)(N + EMU_BN - 1) / EMU_BN * EMU_BN * kpad; P.expT_n += N;
      P.sliceL.push_back(da); E.sliceT.push_back(db);
      EmuSeg sg{};
      sg.a_off = da.out_off; sg.b_off = db.out_off; sg.ea_off = da.exp_off; sg.eb_off = db.exp_off;
      sg.ksteps = kpad / 32; sg.alpha = 1.0; sg.keep = keep;
      E.segs.push_back(sg);
    }
    for (int m0 = 0; m0 < M; m0 += EMU_BM)
      for (int n0 = 0; n0 < N; n0 += EMU_BN) E.tiles.push_back(EmuTile{0, m0, n0, 1});
    E.jobs.push_back(job);
    DevEmu de;
    try {
      upload_emu(P, kappa, de);
      BufTable bt{};
      bt.p[B_OPS_L] = const_cast<double *>(A); bt.p[B_OPS_R] = const_cast<double *>(B); bt.p[B_NEW] = C;
      CK(cudaEventRecord(ev[3], stream));
      run_emu_slice(de, EMU_SLICE_L, bt);
      run_emu_slice(de, 0, bt);
      CK(cudaEventRecord(ev[4], stream));
      run_emu_stage(de, 0, 2, bt, keep != kappa);
      CK(cudaEventRecord(ev[5], stream));
      CK(cudaEventSynchronize(ev[5]));
      float a = 0, b = 0;
      CK(cudaEventElapsedTime(&a, ev[3], ev[4]));
      CK(cudaEventElapsedTime(&b, ev[4], ev[5]));
      if (ms_slice) *ms_slice = a;
      if (ms_gemm) *ms_gemm = b;
    } catch (...) { free_emu(de); throw; }
    free_emu(de);
  }
  // C = sum_g alpha_g A_g B_g in performant mode (reading s21): one segment per class, slice counts set by
  // k_emu_choose exactly as in stage 2 of H_eff.psi; keep_out[g] receives them.
  void emu_sum(int M, int N, int K, int n, const double *A, const double *B, const double *alpha, double *C, int kappa,
               int kmin, int *keep_out) override {
    if (kappa < 2 || kappa > EMU_MAX_KAPPA) throw std::invalid_argument("slices must be in [2, 7]");
    if (M < 1 || N < 1 || K < 1 || K > 16384 || n < 1) throw std::invalid_argument("emu_sum: needs M, N, n >= 1 and 1 <= K <= 16384");
    HeffPlan P;
    P.emu.assign(1, EmuPass());
    EmuPass &E = P.emu[0];
    EmuJob job{};
    job.c = mkref(B_NEW, 0); job.scale = -1; job.n1 = FLAT; job.M = M; job.N = N; job.c_ld = N; job.seg_begin = 0; job.seg_end = n;
    const int kpad = (K + 31) / 32 * 32;
    for (int g = 0; g < n; ++g) {
      EmuSliceDesc da{}, db{};
      da.src = mkref(B_OPS_L, (int64_t)g * M * K); da.mstride = 0; da.lstride = 1; da.linestride = K;
      da.n_members = 1; da.dl = da.dlpad = K; da.lines = M; da.ld = kpad; da.tile_rows = EMU_BM;
      da.out_off = P.emuL_bytes; da.exp_off = P.expL_n;
      P.emuL_bytes += (int64_t)(M + EMU_BM - 1) / EMU_BM * EMU_BM * kpad; P.expL_n += M;
      db.src = mkref(B_OPS_R, (int64_t)g * K * N); db.mstride = 0; db.lstride = N; db.linestride = 1;
      db.n_members = 1; db.dl = db.dlpad = K; db.lines = N; db.ld = kpad; db.tile_rows = EMU_BN;
      db.out_off = P.emuT_bytes; db.exp_off = P.expT_n;
      P.emuT_bytes += (int64_t)(N + EMU_BN - 1) / EMU_BN * EMU_BN * kpad; P.expT_n += N;
      P.sliceL.push_back(da); E.sliceT.push_back(db);
      EmuSeg sg{};
      sg.a_off = da.out_off; sg.b_off = db.out_off; sg.ea_off = da.exp_off; sg.eb_off = db.exp_off;
      sg.ksteps = kpad / 32; sg.alpha = alpha[g]; sg.keep = kappa;
      E.segs.push_back(sg);
    }
    for (int m0 = 0; m0 < M; m0 += EMU_BM)
      for (int n0 = 0; n0 < N; n0 += EMU_BN) E.tiles.push_back(EmuTile{0, m0, n0, 1});
    E.jobs.push_back(job);
    DevEmu de;
    try {
      upload_emu(P, kappa, de);
      BufTable bt{};
      bt.p[B_OPS_L] = const_cast<double *>(A); bt.p[B_OPS_R] = const_cast<double *>(B); bt.p[B_NEW] = C;
      run_emu_slice(de, EMU_SLICE_L, bt);
      run_emu_slice(de, 0, bt);
      run_emu_choose(de, 0, kmin);
      run_emu_stage(de, 0, 2, bt, true);
      std::vector<EmuSeg> back(n);
      download(back.data(), de.pass[0].segs, sizeof(EmuSeg) * n);
      for (int g = 0; g < n; ++g) keep_out[g] = back[g].keep;
    } catch (...) { free_emu(de); throw; }
    free_emu(de);
  }
  // Static schedule of the persistent kernel: jobs by work (k steps + a per-segment drain cost, longest first), each
  // tile given to the least loaded of `grid` CTAs (LPT); the list is regrouped per CTA.  With `gangs` (stage 2) the
  // tiles (m0, n0) of one job -- which walk the same segment list -- are placed on different CTAs at the same start
  // time (the gang waits for its most loaded member) and carry the gang size in EmuTile.work; the kernel's producers
  // then meet at a counter (GangSync in emu_seg.cuh), so an operator tile streamed by one CTA is found in L2 by the
  // CTAs of the other n-tiles and a T tile by those of the other m-tiles.  Every CTA's list follows the one global job
  // order, so the (bounded) waits cannot form a cycle.  the option emu_gang = 0 switches the gangs off.  Returns whether
  // any tile carries a gang.
  bool up_tiles(const std::vector<EmuTile> &tiles, const std::vector<EmuJob> &jobs, const std::vector<EmuSeg> &segs,
                void **d_tiles, void **d_cta, int *grid, bool gangs) {
    const int G = std::max(1, std::min((int)tiles.size(), n_sm));
    std::vector<int64_t> jwork(jobs.size(), 0);
    for (size_t j = 0; j < jobs.size(); ++j)
      for (int sgi = jobs[j].seg_begin; sgi < jobs[j].seg_end; ++sgi) jwork[j] += segs[sgi].ksteps + 6;
    std::vector<std::vector<int>> jtiles(jobs.size());
    for (size_t i = 0; i < tiles.size(); ++i) jtiles[tiles[i].job].push_back((int)i);
    std::vector<int> jorder(jobs.size());
    for (size_t j = 0; j < jorder.size(); ++j) jorder[j] = (int)j;
    std::stable_sort(jorder.begin(), jorder.end(), [&](int x, int y) { return jwork[x] > jwork[y]; });
    std::vector<int64_t> load(G, 0);
    std::vector<int> cta_of(G);
    std::vector<std::vector<EmuTile>> bins(G);
    bool any = false;
    for (int j : jorder) {
      const int T = (int)jtiles[j].size();
      if (T == 0) continue;
      const bool gang = gangs && T >= 2 && T <= G && T <= 16;
      for (int b = 0; b < G; ++b) cta_of[b] = b;
      const int pick = std::min(T, G);
      std::partial_sort(cta_of.begin(), cta_of.begin() + pick, cta_of.end(),
                        [&](int x, int y) { return load[x] != load[y] ? load[x] < load[y] : x < y; });
      if (gang) {
        const int64_t start = load[cta_of[T - 1]];
        for (int i = 0; i < T; ++i) {
          EmuTile t = tiles[jtiles[j][i]]; t.work = T;
          bins[cta_of[i]].push_back(t);
          load[cta_of[i]] = start + jwork[j] + 8;
        }
        any = true;
      } else {
        for (int i = 0; i < T; ++i) {
          const int b = (int)(std::min_element(load.begin(), load.end()) - load.begin());
          EmuTile t = tiles[jtiles[j][i]]; t.work = 0;
          bins[b].push_back(t);
          load[b] += jwork[j] + 8;
        }
      }
    }
    std::vector<EmuTile> grouped;
    std::vector<int> begin(G + 1, 0);
    for (int b = 0; b < G; ++b) {
      grouped.insert(grouped.end(), bins[b].begin(), bins[b].end());
      begin[b + 1] = (int)grouped.size();
    }
    *d_tiles = up(grouped); *d_cta = up(begin); *grid = tiles.empty() ? 0 : G;
    return any;
  }
  // Static schedule of k_emu_s1: items by work (n-tiles x k steps, longest first), each to the least loaded CTA.  The
  // line tiles of one unit have equal work, so they land on different CTAs at about the same time and find each
  // other's psi tiles in L2.
  void up_items(const EmuPass &E, DevEmu::Pass &d) {
    d.n_items1 = (int)E.items1.size();
    if (d.n_items1 == 0) return;
    const int G = std::max(1, std::min(d.n_items1, n_sm));
    std::vector<int> order(E.items1.size());
    for (size_t i = 0; i < order.size(); ++i) order[i] = (int)i;
    auto work = [&](int i) { const EmuS1Item &it = E.items1[i]; return (int64_t)(it.nt_end - it.nt_begin) * (it.ksteps + 2) + 4 * it.ksteps; };
    std::stable_sort(order.begin(), order.end(), [&](int x, int y) { return work(x) > work(y); });
    typedef std::pair<int64_t, int> LB;
    std::priority_queue<LB, std::vector<LB>, std::greater<LB>> pq;
    for (int b = 0; b < G; ++b) pq.push({0, b});
    std::vector<std::vector<EmuS1Item>> bins(G);
    for (int i : order) {
      LB top = pq.top(); pq.pop();
      bins[top.second].push_back(E.items1[i]);
      pq.push({top.first + work(i), top.second});
    }
    std::vector<EmuS1Item> grouped;
    std::vector<int> begin(G + 1, 0);
    for (int b = 0; b < G; ++b) {
      grouped.insert(grouped.end(), bins[b].begin(), bins[b].end());
      begin[b + 1] = (int)grouped.size();
    }
    d.items1 = up(grouped); d.cta_s1 = up(begin); d.ntiles1 = up(E.ntiles1); d.grid_s1 = G;
  }
  void up_slices(const std::vector<EmuSliceDesc> &v, DevEmu::Slices &out) {
    out.n = (int)v.size(); out.max_lines = 0;
    std::vector<int2> work;
    for (size_t i = 0; i < v.size(); ++i) {
      out.max_lines = std::max(out.max_lines, v[i].lines);
      if (v[i].bound == 2) continue;                       // written by the stage-1 epilogue
      for (int l0 = 0; l0 < v[i].lines; l0 += 64) work.push_back(make_int2((int)i, l0));
    }
    out.n_work = (int)work.size();
    out.descs = up(v);
    out.work = up(work);
  }
  void upload_emu(const HeffPlan &P, int kappa, DevEmu &out) override {
    free_emu(out);
    if (kappa < 2 || kappa > 8) throw std::invalid_argument("slices must be in [2, 7]");     // 8: the 3xTF32 engine
    out.kappa = kappa;
    up_slices(P.sliceL, out.sliceL); up_slices(P.sliceR, out.sliceR); up_slices(P.sliceP, out.sliceP);
    out.pass.resize(P.emu.size());
    for (size_t p = 0; p < P.emu.size(); ++p) {
      const EmuPass &E = P.emu[p];
      DevEmu::Pass &d = out.pass[p];
      up_slices(E.sliceT, d.sliceT);
      d.n_tiles1 = (int)E.tiles1.size(); d.segs1 = up(E.segs1); d.jobs1 = up(E.jobs1);
      up_tiles(E.tiles1, E.jobs1, E.segs1, &d.tiles1, &d.cta1, &d.grid1, false);
      up_items(E, d);
      d.n_tiles = (int)E.tiles.size(); d.n_jobs = (int)E.jobs.size(); d.segs = up(E.segs); d.jobs = up(E.jobs);
      if (up_tiles(E.tiles, E.jobs, E.segs, &d.tiles, &d.cta, &d.grid, P.opt.emu_gang != 0))
        d.gang = up(std::vector<int>(E.jobs.size() + 1, 0));
    }
    out.slL = alloc((size_t)kappa * P.emuL_bytes + 64); out.slR = alloc((size_t)kappa * P.emuR_bytes + 64);
    out.slP = alloc((size_t)kappa * P.emuP_bytes + 64); out.slT = alloc((size_t)kappa * P.emuT_bytes + 64);
    out.n_norm_descs = (int)P.emu_norms.size(); out.n_psi = (int)P.psi.size();
    for (auto &nd : P.emu_norms) out.max_norm_lines = std::max(out.max_norm_lines, nd.lines);
    std::vector<EmuPsiDesc> pd;
    for (const PsiBlock &b : P.psi) pd.push_back(EmuPsiDesc{b.off, (int32_t)b.dL, (int32_t)b.dR});
    out.norm_descs = up(P.emu_norms); out.psi_descs = up(pd);
    out.norms = alloc(sizeof(double) * (P.emu_norm_elems + 1));
    out.products = alloc(16);
    CK(cudaMemsetAsync(out.products, 0, 16, stream));
    out.exL = alloc(sizeof(int32_t) * (P.expL_n + 128)); out.exR = alloc(sizeof(int32_t) * (P.expR_n + 128));
    out.exP = alloc(sizeof(int32_t) * (P.expP_n + 128)); out.exT = alloc(sizeof(int32_t) * (P.expT_n + 128));
    CK(cudaStreamSynchronize(stream));
  }
  void free_emu(DevEmu &e) override {
    release(e.sliceL.descs); release(e.sliceR.descs); release(e.sliceP.descs);
    release(e.sliceL.work); release(e.sliceR.work); release(e.sliceP.work);
    for (auto &p : e.pass) {
      release(p.sliceT.descs); release(p.sliceT.work); release(p.segs1); release(p.jobs1); release(p.tiles1); release(p.cta1);
      release(p.segs); release(p.jobs); release(p.tiles); release(p.cta); release(p.gang);
      release(p.items1); release(p.ntiles1); release(p.cta_s1);
    }
    release(e.slL); release(e.slR); release(e.slP); release(e.slT);
    release(e.exL); release(e.exR); release(e.exP); release(e.exT);
    release(e.norm_descs); release(e.psi_descs); release(e.norms); release(e.products);
    e = DevEmu();
  }
  void run_emu_slice(const DevEmu &e, int which, const BufTable &bufs) override {
    const DevEmu::Slices &sd = which == EMU_SLICE_L ? e.sliceL : which == EMU_SLICE_R ? e.sliceR
                               : which == EMU_SLICE_PSI ? e.sliceP : e.pass[which].sliceT;
    if (sd.n_work == 0) return;
    int8_t *sl = (int8_t *)(which == EMU_SLICE_L ? e.slL : which == EMU_SLICE_R ? e.slR : which == EMU_SLICE_PSI ? e.slP : e.slT);
    int32_t *ex = (int32_t *)(which == EMU_SLICE_L ? e.exL : which == EMU_SLICE_R ? e.exR : which == EMU_SLICE_PSI ? e.exP : e.exT);
    const unsigned grid = (unsigned)sd.n_work;
    const EmuSliceDesc *ds = (const EmuSliceDesc *)sd.descs;
    const int2 *wk = (const int2 *)sd.work;
    if (e.kappa == 8) {
      ++n_launches;
      k_tf32_slice_desc<<<grid, 256, 0, stream>>>(ds, wk, bufs, (unsigned char *)sl);
      CK(cudaGetLastError());
      return;
    }
#define EMU_SLICE(KP) case KP: ++n_launches; k_emu_slice_desc<KP><<<grid, 256, 0, stream>>>(ds, wk, bufs, sl, ex, (const double *)e.norms); break;
    switch (e.kappa) { EMU_SLICE(2) EMU_SLICE(3) EMU_SLICE(4) EMU_SLICE(5) EMU_SLICE(6) EMU_SLICE(7) }
#undef EMU_SLICE
    CK(cudaGetLastError());
  }
  void run_emu_norms(const DevEmu &e, int which, const BufTable &bufs) override {
    if (e.n_norm_descs == 0) return;
    ++n_launches;
    if (which < 0)
      k_emu_opnorm<<<dim3((unsigned)e.n_norm_descs, (unsigned)((e.max_norm_lines + 7) / 8)), 256, 0, stream>>>(
          (const EmuNormDesc *)e.norm_descs, bufs, (double *)e.norms);
    else
      k_emu_psinorm<<<e.n_psi, 256, 0, stream>>>((const EmuPsiDesc *)e.psi_descs, bufs.p[B_PSI_IN], (double *)e.norms);
    CK(cudaGetLastError());
  }
  void run_emu_stage(const DevEmu &e, int pass, int stage, const BufTable &bufs, bool performant = false) override {
    const DevEmu::Pass &p = e.pass[pass];
    if (stage == 1 && p.n_items1 > 0 && e.kappa != 8) {
      const int smem1 = s1_smem_bytes(e.kappa);
#define S1_LAUNCH(KP)                                                                                     \
      case KP:                                                                                            \
        CK(cudaFuncSetAttribute(k_emu_s1<KP>, cudaFuncAttributeMaxDynamicSharedMemorySize, smem1));       \
        ++n_launches;                                                                                     \
        k_emu_s1<KP><<<p.grid_s1, S1_THREADS, smem1, stream>>>((const EmuS1Item *)p.items1, (const int *)p.cta_s1, \
            (const EmuS1Tile *)p.ntiles1, (const EmuJob *)p.jobs1, bufs, (const int8_t *)e.slR, (const int8_t *)e.slP, \
            (const int32_t *)e.exR, (const int32_t *)e.exP, (int8_t *)e.slT, (int32_t *)e.exT, (const double *)e.norms); \
        break;
      switch (e.kappa) { S1_LAUNCH(2) S1_LAUNCH(3) S1_LAUNCH(4) S1_LAUNCH(5) S1_LAUNCH(6) S1_LAUNCH(7) }
#undef S1_LAUNCH
      CK(cudaGetLastError());
    }
    const int n_tiles = stage == 1 ? p.n_tiles1 : p.n_tiles;
    if (n_tiles == 0) return;
    const EmuJob *jobs = (const EmuJob *)(stage == 1 ? p.jobs1 : p.jobs);
    const EmuSeg *segs = (const EmuSeg *)(stage == 1 ? p.segs1 : p.segs);
    const EmuTile *tiles = (const EmuTile *)(stage == 1 ? p.tiles1 : p.tiles);
    const int8_t *sa = (const int8_t *)(stage == 1 ? e.slR : e.slL), *sb = (const int8_t *)(stage == 1 ? e.slP : e.slT);
    const int32_t *ea = (const int32_t *)(stage == 1 ? e.exR : e.exL), *eb = (const int32_t *)(stage == 1 ? e.exP : e.exT);
    const int grid = stage == 1 ? p.grid1 : p.grid;
    const int *cta = (const int *)(stage == 1 ? p.cta1 : p.cta);
    int *gang = stage == 1 ? nullptr : (int *)p.gang;
    const int epoch = gang ? ++p.epoch : 0;
    if (e.kappa == 8) {
      const int smem3 = TF32_STAGES * TF32_STAGE + EMU_BM * 33 * 8;
      CK(cudaFuncSetAttribute(k_tf32_seg, cudaFuncAttributeMaxDynamicSharedMemorySize, smem3));
      ++n_launches;
      k_tf32_seg<<<grid, TF32_THREADS, smem3, stream>>>(jobs, segs, tiles, cta, bufs, (const unsigned char *)sa, (const unsigned char *)sb,
                                                       (unsigned char *)e.slT, gang, epoch);
      CK(cudaGetLastError());
      return;
    }
    const int smem = EMU_STAGES * e.kappa * (2 * EMU_BM * 16 + 2 * EMU_BN * 16) + EMU_BM * 33 * 8;
#define EMU_LAUNCH2(KP, PF)                                                                              \
      CK(cudaFuncSetAttribute(k_emu_seg<KP, PF>, cudaFuncAttributeMaxDynamicSharedMemorySize, smem));    \
      ++n_launches;                                                                                      \
      k_emu_seg<KP, PF><<<grid, EMU_THREADS, smem, stream>>>(jobs, segs, tiles, cta, bufs, sa, sb, ea, eb, \
          (int8_t *)e.slT, (int32_t *)e.exT, (const double *)e.norms, gang, epoch);
#define EMU_LAUNCH(KP)                                                                                   \
    case KP:                                                                                             \
      if (performant && stage == 2) { EMU_LAUNCH2(KP, true) } else { EMU_LAUNCH2(KP, false) }            \
      break;
    switch (e.kappa) { EMU_LAUNCH(2) EMU_LAUNCH(3) EMU_LAUNCH(4) EMU_LAUNCH(5) EMU_LAUNCH(6) EMU_LAUNCH(7) }
#undef EMU_LAUNCH
#undef EMU_LAUNCH2
    CK(cudaGetLastError());
  }
  void run_emu_choose(const DevEmu &e, int pass, int kmin) override {
    const DevEmu::Pass &p = e.pass[pass];
    if (p.n_tiles == 0 || p.n_jobs == 0 || e.kappa == 8) return;
    ++n_launches;
    k_emu_choose<<<p.n_jobs, 128, 0, stream>>>((const EmuJob *)p.jobs, (EmuSeg *)p.segs, (const int32_t *)e.exL,
                                               (const int32_t *)e.exT, e.kappa, kmin, (unsigned long long *)e.products);
    CK(cudaGetLastError());
  }
  void reset_emu_products(const DevEmu &e) override {
    if (e.products) CK(cudaMemsetAsync(e.products, 0, 16, stream));
  }
  void emu_products(const DevEmu &e, uint64_t out[2]) override {
    out[0] = out[1] = 0;
    if (e.products) download(out, e.products, 16);
  }
  uint64_t n_launches = 0;                                   // kernels launched by this backend so far (bench.py gpu_launches)
  uint64_t launch_count() override { return n_launches; }
  void timer_mark(int slot) override { CK(cudaEventRecord(ev[slot], stream)); }
  double timer_ms(int a, int b) override {
    CK(cudaEventSynchronize(ev[b]));
    float ms = 0;
    CK(cudaEventElapsedTime(&ms, ev[a], ev[b]));
    return ms;
  }
  // INT8 tensor pipe: check one tcgen05 s8 MMA (and an accumulating sequence) element by element against the
  // integer definition, then time back-to-back 128 x 256 x 32 MMAs on every SM.
  double measure_peak_i8() {
    const int M = 128, N = 256, K = 32;
    int32_t *out = (int32_t *)alloc(sizeof(int32_t) * M * N);
    std::vector<int32_t> host(M * N);
    for (int n_mma : {1, 5}) {
      k_peak_i8<256><<<1, 128, 0, stream>>>(n_mma, out);
      CK(cudaGetLastError());
      download(host.data(), out, sizeof(int32_t) * M * N);
      const int reps = (n_mma + 1) / 2;       // accumulator 0 receives MMAs 0, 2, 4, ...
      for (int m = 0; m < M; ++m)
        for (int n = 0; n < N; ++n) {
          int ref = 0;
          for (int k = 0; k < K; ++k) ref += (((3 * m + 5 * k) % 11) - 5) * (((7 * n + k) % 9) - 4);
          if (host[(size_t)m * N + n] != ref * reps) {
            release(out);
            throw std::runtime_error("tcgen05 kind::i8 self-check failed at (" + std::to_string(m) + "," +
                                     std::to_string(n) + "): got " + std::to_string(host[(size_t)m * N + n]) +
                                     ", expected " + std::to_string(ref * reps));
          }
        }
    }
    release(out);
    const int n_mma = 20000;
    k_peak_i8<256><<<n_sm, 128, 0, stream>>>(2000, nullptr);   // warm-up
    double best = 0;
    for (int rep = 0; rep < 3; ++rep) {
      CK(cudaEventRecord(ev[6], stream));
      k_peak_i8<256><<<n_sm, 128, 0, stream>>>(n_mma, nullptr);
      CK(cudaEventRecord(ev[7], stream));
      CK(cudaEventSynchronize(ev[7]));
      float ms = 0;
      CK(cudaEventElapsedTime(&ms, ev[6], ev[7]));
      best = std::max(best, 2.0 * M * N * K * n_mma * n_sm / (ms * 1e-3));
    }
    return best;
  }
  // TF32 tensor pipe: 5 accumulating 128 x 256 x 8 MMAs of A = 1, B = 0.5 must give 3 * 4 = 12 in accumulator 0
  // (MMAs 0, 2, 4), then back-to-back MMAs are timed on every SM.
  double measure_peak_tf32() {
    float *out = (float *)alloc(sizeof(float) * 128);
    float host[128];
    k_peak_tf32<<<1, 128, 0, stream>>>(5, out);
    CK(cudaGetLastError());
    download(host, out, sizeof(host));
    release(out);
    for (int i = 0; i < 128; ++i)
      if (host[i] != 12.0f) throw std::runtime_error("tcgen05 kind::tf32 self-check failed: got " + std::to_string(host[i]) + ", expected 12");
    const int n_mma = 20000;
    k_peak_tf32<<<n_sm, 128, 0, stream>>>(2000, nullptr);
    double best = 0;
    for (int rep = 0; rep < 3; ++rep) {
      CK(cudaEventRecord(ev[6], stream));
      k_peak_tf32<<<n_sm, 128, 0, stream>>>(n_mma, nullptr);
      CK(cudaEventRecord(ev[7], stream));
      CK(cudaEventSynchronize(ev[7]));
      float ms = 0;
      CK(cudaEventElapsedTime(&ms, ev[6], ev[7]));
      best = std::max(best, 2.0 * 128 * 256 * 8 * n_mma * n_sm / (ms * 1e-3));
    }
    return best;
  }
  // FP64 vector (non-tensor) FMA rate: the unit the emulated epilogue recombines on (8 independent chains per thread)
  double measure_peak_dfma() {
    double *sink = (double *)alloc(8);
    const int iters = 4096, blocks = n_sm * 4, threads = 256;
    k_peak_dfma<<<blocks, threads, 0, stream>>>(64, sink, 1.0);   // warm-up
    double best = 0;
    for (int rep = 0; rep < 3; ++rep) {
      CK(cudaEventRecord(ev[6], stream));
      k_peak_dfma<<<blocks, threads, 0, stream>>>(iters, sink, 1.0);
      CK(cudaEventRecord(ev[7], stream));
      CK(cudaEventSynchronize(ev[7]));
      float ms = 0;
      CK(cudaEventElapsedTime(&ms, ev[6], ev[7]));
      best = std::max(best, 2.0 * 8 * iters * (double)threads * blocks / (ms * 1e-3));
    }
    release(sink);
    return best;
  }
  double measure_peak(int which) override {
    if (which == 1) return measure_peak_i8();
    if (which == 2) return measure_peak_tf32();
    if (which == 3) return measure_peak_dfma();
    if (which != 0) throw std::runtime_error("peak measurement for this mode is not implemented");
    double *sink = (double *)alloc(8);
    const int iters = 20000, blocks = n_sm * 4, threads = 256;
    k_peak_dmma<<<blocks, threads, 0, stream>>>(200, sink);   // warm-up
    double best = 0;
    for (int rep = 0; rep < 3; ++rep) {
      CK(cudaEventRecord(ev[6], stream));
      k_peak_dmma<<<blocks, threads, 0, stream>>>(iters, sink);
      CK(cudaEventRecord(ev[7], stream));
      CK(cudaEventSynchronize(ev[7]));
      float ms = 0;
      CK(cudaEventElapsedTime(&ms, ev[6], ev[7]));
      double flops = 512.0 * 16 * iters * (threads / 32) * blocks;
      best = std::max(best, flops / (ms * 1e-3));
    }
    release(sink);
    return best;
  }
};

// ------------------------------------------------------------------ allocation-free entry point (dmrg_dots_noalloc)
// Scratch of the dot-product kernels for callers that may not allocate (CUDA graph capture, serving loops): the
// per-block partial sums live in a file-scope device array instead of the backend's cudaMalloc'ed buffer.  Every
// GPU that loads the library holds these 74 KB until exit.  In host code `g_dots_scratch` is a host-side stand-in,
// NOT a device address: the address is taken once per device with cudaGetSymbolAddress (noalloc_scratch) and that
// pointer is what the kernels receive.
static __device__ __align__(256) double g_dots_scratch[DOT_BLOCKS * MAX_BASIS];
static const int NOALLOC_MAX_DEVICES = 64;
static double *g_dots_scratch_ptr[NOALLOC_MAX_DEVICES];     // per device, filled on first use (null = not yet)
static thread_local char g_noalloc_err[256];

static cudaError_t noalloc_scratch(int dev, double **out) {
  // racing first calls on one device both write the same value
  double *p = __atomic_load_n(&g_dots_scratch_ptr[dev], __ATOMIC_ACQUIRE);
  if (!p) {
    cudaError_t e = cudaGetSymbolAddress((void **)&p, g_dots_scratch);    // device `dev` is current (checked by the caller)
    if (e != cudaSuccess) return e;
    __atomic_store_n(&g_dots_scratch_ptr[dev], p, __ATOMIC_RELEASE);
  }
  *out = p;
  return cudaSuccess;
}

Backend *make_cuda_backend(int device, void *stream, std::string *err) {
  try {
    int n = 0;
    cudaError_t e = cudaGetDeviceCount(&n);
    if (e != cudaSuccess || n == 0) {
      cudaGetLastError();
      *err = "no CUDA device available (there is no CPU fallback)";
      return nullptr;
    }
    if (device >= n) { *err = "device ordinal out of range"; return nullptr; }
    return new CudaBackend(device, stream);
  } catch (const std::exception &ex) {
    *err = ex.what();
    return nullptr;
  }
}

}  // namespace dmrg

extern "C" {
const char *dmrg_noalloc_last_error(void) { return dmrg::g_noalloc_err; }

int dmrg_dots_noalloc(void *cuda_stream, const double *V_dev, int64_t ld, int nvec, const double *w_dev, int64_t n,
                      double *out_dev) {
  using namespace dmrg;
  auto fail = [](int code, const char *msg) { snprintf(g_noalloc_err, sizeof g_noalloc_err, "%s", msg); return code; };
  if (!V_dev || !w_dev || !out_dev || n < 0 || ld < 0) return fail(-1, "dmrg_dots_noalloc: null pointer or negative size");
  if (nvec < 1 || nvec > MAX_BASIS) {
    snprintf(g_noalloc_err, sizeof g_noalloc_err,
             "dmrg_dots_noalloc: nvec = %d is outside [1, %d], the capacity of the static scratch (%d x %d doubles)", nvec,
             MAX_BASIS, MAX_BASIS, DOT_BLOCKS);
    return -1;
  }
  int dev = -1;
  cudaError_t e = cudaGetDevice(&dev);
  if (e != cudaSuccess) return fail(-4, cudaGetErrorString(e));
  if (dev < 0 || dev >= NOALLOC_MAX_DEVICES) return fail(-5, "dmrg_dots_noalloc: device ordinal beyond the per-device table");
  double *scratch = nullptr;
  e = noalloc_scratch(dev, &scratch);
  if (e != cudaSuccess) return fail(-4, cudaGetErrorString(e));
  // every entry of the scratch that k_dots_final reads (nvec x DOT_BLOCKS) is overwritten by k_dots_partial first, so
  // nothing has to start at zero although the array keeps the last call's contents
  cudaStream_t st = (cudaStream_t)cuda_stream;
  k_dots_partial<<<DOT_BLOCKS, DOT_THREADS, 0, st>>>(V_dev, ld, nvec, w_dev, n, scratch);
  k_dots_final<<<nvec, 32, 0, st>>>(scratch, DOT_BLOCKS, out_dev);
  e = cudaGetLastError();
  if (e != cudaSuccess) return fail(-4, cudaGetErrorString(e));
  g_noalloc_err[0] = 0;
  return 0;
}
}  // extern "C"
