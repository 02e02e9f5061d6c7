// Device backend interface: memory, descriptor upload and the kernels of kernels.cu.
// The product has exactly one implementation (CUDA, sm_100a); there is no CPU path.
#pragma once
#include "internal.h"

namespace dmrg {

struct DevJobList {           // device-resident copy of a JobList
  void *jobs = nullptr, *segs = nullptr, *tiles = nullptr;
  int n_jobs = 0, n_segs = 0, n_tiles = 0;
  int tile = 32;              // CTA tile edge the list was tiled for (32, 48, 64)
  int role = 0;               // which phase the list belongs to (names the kernel instantiation)
  int64_t flops = 0;
};
struct DevDiag { void *jobs = nullptr, *terms = nullptr; int n_jobs = 0; };
struct DevReduce { void *jobs = nullptr; int n_jobs = 0; };

struct DevEmu {               // device side of the emulated mode (HeffPlan::sliceL / sliceR / sliceP / emu)
  struct Slices { void *descs = nullptr, *work = nullptr; int n = 0, max_lines = 0, n_work = 0; };   // work: int2 (descriptor, line0) per 64-line tile
  struct Pass { Slices sliceT;
                // per stage: descriptors, the tile list grouped per CTA and cta_begin[grid + 1]
                void *segs1 = nullptr, *jobs1 = nullptr, *tiles1 = nullptr, *cta1 = nullptr; int n_tiles1 = 0, grid1 = 0;
                void *segs = nullptr, *jobs = nullptr, *tiles = nullptr, *cta = nullptr; int n_tiles = 0, grid = 0, n_jobs = 0;
                // second-generation stage 1 (emu_s1.cuh): work items grouped per CTA, n-tile list
                void *items1 = nullptr, *ntiles1 = nullptr, *cta_s1 = nullptr; int n_items1 = 0, grid_s1 = 0;
                // stage-2 gangs (tiles of one job started together, see up_tiles): arrival counters per job, launches so far
                void *gang = nullptr; mutable int epoch = 0; };
  Slices sliceL, sliceR, sliceP;
  std::vector<Pass> pass;
  // int8 slice buffers and int32 exponents: left operators, right operators, psi, T
  void *slL = nullptr, *slR = nullptr, *slP = nullptr, *slT = nullptr;
  void *exL = nullptr, *exR = nullptr, *exP = nullptr, *exT = nullptr;
  void *norm_descs = nullptr, *psi_descs = nullptr, *norms = nullptr;    // bound exponents of T
  int n_norm_descs = 0, n_psi = 0, max_norm_lines = 0;
  int kappa = 0;                                                            // slice count the buffers hold
  void *products = nullptr;             // performant mode: two 64-bit counters (slice products x k steps x tiles: kept, eager)
};
enum { EMU_SLICE_L = -1, EMU_SLICE_R = -2, EMU_SLICE_PSI = -3 };           // `which` of run_emu_slice (>= 0: T of a pass)

struct BufTable { double *p[N_BUFS]; };

class Backend {
 public:
  virtual ~Backend() {}
  virtual void make_current() = 0;                       // cudaSetDevice(the backend's device) if another one is current
  virtual void *alloc(size_t bytes) = 0;                 // throws std::bad_alloc / runtime_error
  virtual void release(void *p) = 0;
  virtual void upload(void *dst, const void *src, size_t bytes) = 0;     // host -> device, stream ordered
  virtual void download(void *dst, const void *src, size_t bytes) = 0;   // device -> host, synchronises
  virtual void copy(void *dst, const void *src, size_t bytes) = 0;       // device -> device
  virtual void zero(void *dst, size_t bytes) = 0;
  virtual void sync() = 0;
  virtual void upload_jobs(const JobList &jl, DevJobList &out, int role) = 0;
  virtual void free_jobs(DevJobList &jl) = 0;
  virtual void upload_diag(const std::vector<DiagJob> &jobs, const std::vector<DiagTerm> &terms, DevDiag &out) = 0;
  virtual void free_diag(DevDiag &d) = 0;
  virtual void upload_reduce(const std::vector<ReduceJob> &jobs, DevReduce &out) = 0;
  virtual void free_reduce(DevReduce &d) = 0;
  virtual void run_reduce(const DevReduce &d, const double *partial, double *out) = 0;
  // C = colscale * sum_seg alpha A B for every tile of the list (FP64 tensor pipe)
  virtual void run_jobs(const DevJobList &jl, const BufTable &bufs) = 0;
  virtual void run_diag(const DevDiag &d, const BufTable &bufs, double *out) = 0;
  // Davidson vector work; every scalar stays on the device
  virtual void dots(const double *V, int64_t ld, int nvec, const double *w, int64_t n, double *out) = 0;
  virtual void davidson_small(double *G, int ldg, int m, const double *col, double *y, double *theta_out) = 0;
  virtual void ritz_residual(const double *V, const double *W, int64_t ld, int m, int64_t n, const double *y,
                             const double *theta, double *x, double *r) = 0;
  virtual void precondition(const double *r, const double *diag, const double *theta, double *t, int64_t n) = 0;
  virtual void subtract_projection(const double *V, int64_t ld, int m, const double *c, double *t, int64_t n) = 0;
  virtual void scale_inv_norm(const double *src, const double *nrm2, double *dst, int64_t n) = 0;
  // Ozaki-emulated FP64 GEMM on the INT8 tensor cores (emu.cuh): C[M][N] = A[M][K] B[K][N], row-major device
  // arrays; returns the device time of the tcgen05 kernel (ms_gemm) and of the slicing (ms_slice)
  virtual void tf32_split_run(const double *src, int64_t n, uint32_t *hi, uint32_t *lo) = 0;
  virtual void emu_gemm(int M, int N, int K, const double *A, const double *B, double *C, int kappa, int keep,
                        double *ms_slice, double *ms_gemm) = 0;
  virtual void emu_sum(int M, int N, int K, int n, const double *A, const double *B, const double *alpha, double *C,
                       int kappa, int kmin, int *keep_out) = 0;
  // slice `lines` lines of length K (element (line, k) at src[line * ls + k * ks]) into out[kappa][lines][K] / expo
  virtual void emu_slice(const double *src, int lines, int K, int64_t ls, int64_t ks, int kappa, signed char *out,
                         int *expo) = 0;
  // emulated mode (emu_seg.cuh): descriptors + buffers for `kappa` slices; run_emu_slice slices the left or right
  // operators, psi (EMU_SLICE_*) or the T of pass `which`; run_emu_stage runs the tcgen05 jobs of stage 1 or 2 of a pass
  virtual void upload_emu(const HeffPlan &P, int kappa, DevEmu &out) = 0;
  virtual void free_emu(DevEmu &e) = 0;
  virtual void run_emu_slice(const DevEmu &e, int which, const BufTable &bufs) = 0;
  // line norms behind the bound exponents: which = -1 right-operator norms (per bond), 0 psi norms (per apply)
  virtual void run_emu_norms(const DevEmu &e, int which, const BufTable &bufs) = 0;
  virtual void run_emu_stage(const DevEmu &e, int pass, int stage, const BufTable &bufs, bool performant = false) = 0;
  // performant mode (reading s21): set EmuSeg::keep of the pass's stage-2 segments from the exponents on the device;
  // emu_products: the counters accumulated by run_emu_choose since the last reset (synchronises)
  virtual void run_emu_choose(const DevEmu &e, int pass, int kmin) = 0;
  virtual void reset_emu_products(const DevEmu &e) = 0;
  virtual void emu_products(const DevEmu &e, uint64_t out[2]) = 0;
  virtual uint64_t launch_count() = 0;        // kernels launched so far (micro-benchmarks of measure_peak excluded)
  virtual void timer_mark(int slot) = 0;                 // record a CUDA event on the stream
  virtual double timer_ms(int a, int b) = 0;             // synchronises
  virtual double measure_peak(int which) = 0;            // operations per second of a full-tile micro-kernel
};

Backend *make_cuda_backend(int device, void *stream, std::string *err);

}  // namespace dmrg
