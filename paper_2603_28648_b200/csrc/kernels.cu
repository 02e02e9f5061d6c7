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
#include <new>
#include <stdexcept>
#include <string>
#include <vector>

#include "backend.h"

namespace dmrg {

#define CK(call)                                                                          \
  do {                                                                                    \
    cudaError_t e_ = (call);                                                              \
    if (e_ != cudaSuccess)                                                                \
      throw std::runtime_error(std::string("CUDA: ") + cudaGetErrorString(e_) + " at " #call); \
  } while (0)

static constexpr int FLATV = 1 << 30;
static constexpr int64_t REF_MASK = (1LL << 48) - 1;

__device__ __forceinline__ const double *rd_ref(const BufTable &b, ref_t r) {
  return b.p[r >> 48] + (r & REF_MASK);
}
__device__ __forceinline__ void dmma884(double &d0, double &d1, double a, double b) {
  asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};\n"
               : "+d"(d0), "+d"(d1) : "d"(a), "d"(b));
}

// MT = 8x8 MMA tiles per warp per dimension; 4 warps (2 x 2); CTA tile = (16 MT) x (16 MT); BK = 16.
template <int MT>
__global__ void __launch_bounds__(128) k_gemm_f64(const JobDesc *__restrict__ jobs,
                                                  const SegDesc *__restrict__ segs,
                                                  const TileDesc *__restrict__ tiles, BufTable bufs) {
  constexpr int BM = 16 * MT, BN = 16 * MT, BK = 16;
  constexpr int EA = BM * BK / 128, EB = BK * BN / 128;
  __shared__ double As[2][BM * BK];
  __shared__ double Bs[2][BK * BN];

  const TileDesc td = tiles[blockIdx.x];
  const JobDesc jd = jobs[td.job];
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5, wm = warp & 1, wn = warp >> 1;
  const int m0 = td.m0, n0 = td.n0;
  const int Mrem = jd.M - m0, Nrem = jd.N - n0;   // > 0

  double acc[MT][MT][2];
#pragma unroll
  for (int i = 0; i < MT; ++i)
#pragma unroll
    for (int j = 0; j < MT; ++j) acc[i][j][0] = acc[i][j][1] = 0.0;

  // number of 8-row / 8-column MMA tiles of this warp that hold real data
  int mi_valid = (Mrem - wm * 8 * MT + 7) / 8; mi_valid = max(0, min(MT, mi_valid));
  int nj_valid = (Nrem - wn * 8 * MT + 7) / 8; nj_valid = max(0, min(MT, nj_valid));

  // decomposition of this thread's B columns under both load mappings (fixed per tile)
  const int n1 = jd.n1;
  int nqK[EB], nrK[EB];              // k-contiguous mapping: columns tid/16 + 8 j
#pragma unroll
  for (int j = 0; j < EB; ++j) {
    int n = n0 + (tid >> 4) + 8 * j;
    nqK[j] = n / n1; nrK[j] = n - nqK[j] * n1;
  }
  const int nN = n0 + (tid % BN);    // n-contiguous mapping: one column
  const int nqN = nN / n1, nrN = nN - nqN * n1;

  int seg = jd.seg_begin;
  const int seg_end = jd.seg_end;
  double ra[EA], rb[EB];
  int layA[2], layB[2];              // 0: k fastest in smem rows ([m][k] / [n][k]); 1: [k][m] / [k][n]

  // Global -> registers for (segment s, k offset k0); returns the two layout flags.
  auto load_tile = [&](int s, int k0, int &la, int &lb) {
    const SegDesc sd = segs[s];
    const double *A = rd_ref(bufs, sd.a), *B = rd_ref(bufs, sd.b);
    la = (sd.a_ms == 1 && sd.a_klo != 1) ? 1 : 0;
    lb = (sd.b_nlo == 1 && sd.b_ks != 1) ? 1 : 0;
    if (la == 0) {       // threads run along k
      int k = k0 + (tid & 15);
      int kq = k / sd.a_kn1, kr = k - kq * sd.a_kn1;
      const double *p = A + (int64_t)kq * sd.a_khi + (int64_t)kr * sd.a_klo;
      bool kok = k < sd.K;
#pragma unroll
      for (int j = 0; j < EA; ++j) {
        int mm = (tid >> 4) + 8 * j;
        ra[j] = (kok && mm < Mrem) ? __ldg(p + (int64_t)(m0 + mm) * sd.a_ms) * sd.alpha : 0.0;
      }
    } else {             // threads run along m
      int mm = tid % BM;
      const double *p = A + (int64_t)(m0 + mm) * sd.a_ms;
      bool mok = mm < Mrem;
#pragma unroll
      for (int j = 0; j < EA; ++j) {
        int k = k0 + tid / BM + (128 / BM) * j;
        int kq = k / sd.a_kn1, kr = k - kq * sd.a_kn1;
        ra[j] = (mok && k < sd.K) ? __ldg(p + (int64_t)kq * sd.a_khi + (int64_t)kr * sd.a_klo) * sd.alpha : 0.0;
      }
    }
    if (lb == 0) {       // threads run along k
      int k = k0 + (tid & 15);
      const double *p = B + (int64_t)k * sd.b_ks;
      bool kok = k < sd.K;
#pragma unroll
      for (int j = 0; j < EB; ++j) {
        int nn = (tid >> 4) + 8 * j;
        rb[j] = (kok && nn < Nrem) ? __ldg(p + (int64_t)nqK[j] * sd.b_nhi + (int64_t)nrK[j] * sd.b_nlo) : 0.0;
      }
    } else {             // threads run along n
      const double *p = B + (int64_t)nqN * sd.b_nhi + (int64_t)nrN * sd.b_nlo;
      bool nok = (tid % BN) < Nrem;
#pragma unroll
      for (int j = 0; j < EB; ++j) {
        int k = k0 + tid / BN + (128 / BN) * j;
        rb[j] = (nok && k < sd.K) ? __ldg(p + (int64_t)k * sd.b_ks) : 0.0;
      }
    }
  };
  auto store_tile = [&](int buf, int la, int lb) {
    double *as = As[buf], *bs = Bs[buf];
    if (la == 0) {
      int kk = tid & 15;
#pragma unroll
      for (int j = 0; j < EA; ++j) { int mm = (tid >> 4) + 8 * j; as[mm * BK + (kk ^ (4 * (mm & 3)))] = ra[j]; }
    } else {
      int mm = tid % BM;
#pragma unroll
      for (int j = 0; j < EA; ++j) { int kk = tid / BM + (128 / BM) * j; as[kk * BM + (mm ^ (4 * (kk & 3)))] = ra[j]; }
    }
    if (lb == 0) {
      int kk = tid & 15;
#pragma unroll
      for (int j = 0; j < EB; ++j) { int nn = (tid >> 4) + 8 * j; bs[nn * BK + (kk ^ (4 * (nn & 3)))] = rb[j]; }
    } else {
      int nn = tid % BN;
#pragma unroll
      for (int j = 0; j < EB; ++j) { int kk = tid / BN + (128 / BN) * j; bs[kk * BN + (nn ^ (4 * (kk & 3)))] = rb[j]; }
    }
  };

  if (seg < seg_end) {
    int k0 = 0, K = segs[seg].K, buf = 0;
    load_tile(seg, 0, layA[0], layB[0]);
    store_tile(0, layA[0], layB[0]);
    __syncthreads();
    while (true) {
      // next (segment, k0)
      int nseg = seg, nk0 = k0 + BK;
      if (nk0 >= K) { nseg = seg + 1; nk0 = 0; }
      bool more = nseg < seg_end;
      if (more) load_tile(nseg, nk0, layA[buf ^ 1], layB[buf ^ 1]);
      // compute on the current buffer
      const double *as = As[buf], *bs = Bs[buf];
      const int la = layA[buf], lb = layB[buf];
      const int r = lane >> 2, c = lane & 3;
#pragma unroll
      for (int ks = 0; ks < BK / 4; ++ks) {
        const int k = ks * 4 + c;
        double af[MT], bf[MT];
#pragma unroll
        for (int i = 0; i < MT; ++i) {
          int m = wm * 8 * MT + i * 8 + r;
          af[i] = la == 0 ? as[m * BK + (k ^ (4 * (m & 3)))] : as[k * BM + (m ^ (4 * c))];
        }
#pragma unroll
        for (int j = 0; j < MT; ++j) {
          int n = wn * 8 * MT + j * 8 + r;
          bf[j] = lb == 0 ? bs[n * BK + (k ^ (4 * (n & 3)))] : bs[k * BN + (n ^ (4 * c))];
        }
#pragma unroll
        for (int i = 0; i < MT; ++i)
#pragma unroll
          for (int j = 0; j < MT; ++j)
            if (i < mi_valid && j < nj_valid) dmma884(acc[i][j][0], acc[i][j][1], af[i], bf[j]);
      }
      if (!more) break;
      store_tile(buf ^ 1, layA[buf ^ 1], layB[buf ^ 1]);
      __syncthreads();
      buf ^= 1;
      if (nseg != seg) { seg = nseg; K = segs[seg].K; }
      k0 = nk0;
    }
  }

  // epilogue: one write per element, optional per-column-group scale
  double *C = const_cast<double *>(rd_ref(bufs, jd.c));
  const double *scale = jd.scale >= 0 ? rd_ref(bufs, jd.scale) : nullptr;
#pragma unroll
  for (int i = 0; i < MT; ++i) {
    int mm = wm * 8 * MT + i * 8 + (lane >> 2);
    if (mm >= Mrem) continue;
#pragma unroll
    for (int j = 0; j < MT; ++j) {
#pragma unroll
      for (int e = 0; e < 2; ++e) {
        int nn = wn * 8 * MT + j * 8 + 2 * (lane & 3) + e;
        if (nn >= Nrem) continue;
        int n = n0 + nn;
        int nq = n / n1, nr = n - nq * n1;
        double v = acc[i][j][e];
        if (scale) v *= __ldg(scale + nq);
        C[(int64_t)(m0 + mm) * jd.c_ms + (int64_t)nq * jd.c_nhi + (int64_t)nr * jd.c_nlo] = v;
      }
    }
  }
}

// a7: diag(H_eff)[l][r] = sum_t f_t diag(O_L,t)[l] diag(O_R,t)[r], one CTA per psi block.
__global__ void __launch_bounds__(256) k_heff_diag(const DiagJob *__restrict__ jobs,
                                                   const DiagTerm *__restrict__ terms, BufTable bufs,
                                                   double *__restrict__ out) {
  const DiagJob j = jobs[blockIdx.x];
  const int nel = j.dL * j.dR;
  for (int e = threadIdx.x; e < nel; e += blockDim.x) {
    int l = e / j.dR, r = e - l * j.dR;
    double s = 0.0;
    for (int t = j.t_begin; t < j.t_end; ++t) {
      const DiagTerm dt = terms[t];
      s += dt.f * __ldg(rd_ref(bufs, dt.l) + (int64_t)l * dt.ls) * __ldg(rd_ref(bufs, dt.r) + (int64_t)r * dt.rs);
    }
    out[j.off + e] = s;
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
  cudaEvent_t ev[8];
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
  }
  ~CudaBackend() override {
    cudaFree(dot_partial);
    for (auto &e : ev) cudaEventDestroy(e);
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
  void upload_jobs(const JobList &jl, DevJobList &out) override {
    free_jobs(out);
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

  void run_jobs(const DevJobList &jl, const BufTable &bufs) override {
    if (jl.n_tiles == 0) return;
    k_gemm_f64<2><<<jl.n_tiles, 128, 0, stream>>>((const JobDesc *)jl.jobs, (const SegDesc *)jl.segs,
                                                  (const TileDesc *)jl.tiles, bufs);
    CK(cudaGetLastError());
  }
  void run_diag(const DevDiag &d, const BufTable &bufs, double *out) override {
    if (d.n_jobs == 0) return;
    k_heff_diag<<<d.n_jobs, 256, 0, stream>>>((const DiagJob *)d.jobs, (const DiagTerm *)d.terms, bufs, out);
    CK(cudaGetLastError());
  }
  int vec_blocks(int64_t n) const { return (int)std::max<int64_t>(1, std::min<int64_t>((n + 255) / 256, 4 * n_sm)); }
  void dots(const double *V, int64_t ld, int nvec, const double *w, int64_t n, double *out) override {
    if (nvec > MAX_BASIS) throw std::runtime_error("too many basis vectors");
    k_dots_partial<<<DOT_BLOCKS, DOT_THREADS, 0, stream>>>(V, ld, nvec, w, n, dot_partial);
    k_dots_final<<<nvec, 32, 0, stream>>>(dot_partial, DOT_BLOCKS, out);
    CK(cudaGetLastError());
  }
  void davidson_small(double *G, int ldg, int m, const double *col, double *y, double *theta_out) override {
    if (m > MAX_BASIS) throw std::runtime_error("Davidson basis too large");
    k_davidson_small<<<1, 32, 0, stream>>>(G, ldg, m, col, y, theta_out);
    CK(cudaGetLastError());
  }
  void ritz_residual(const double *V, const double *W, int64_t ld, int m, int64_t n, const double *y,
                     const double *theta, double *x, double *r) override {
    k_ritz_residual<<<vec_blocks(n), 256, 0, stream>>>(V, W, ld, m, n, y, theta, x, r);
    CK(cudaGetLastError());
  }
  void precondition(const double *r, const double *diag, const double *theta, double *t, int64_t n) override {
    k_precondition<<<vec_blocks(n), 256, 0, stream>>>(r, diag, theta, t, n);
    CK(cudaGetLastError());
  }
  void subtract_projection(const double *V, int64_t ld, int m, const double *c, double *t, int64_t n) override {
    k_subtract_projection<<<vec_blocks(n), 256, 0, stream>>>(V, ld, m, c, t, n);
    CK(cudaGetLastError());
  }
  void scale_inv_norm(const double *src, const double *nrm2, double *dst, int64_t n) override {
    k_scale_inv_norm<<<vec_blocks(n), 256, 0, stream>>>(src, nrm2, dst, n);
    CK(cudaGetLastError());
  }
  void timer_mark(int slot) override { CK(cudaEventRecord(ev[slot], stream)); }
  double timer_ms(int a, int b) override {
    CK(cudaEventSynchronize(ev[b]));
    float ms = 0;
    CK(cudaEventElapsedTime(&ms, ev[a], ev[b]));
    return ms;
  }
  double measure_peak(int which) override {
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
