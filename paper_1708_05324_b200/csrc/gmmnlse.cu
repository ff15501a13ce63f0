// Host side of the C ABI declared in include/gmmnlse.h: plan precompute (fp64), the MPA driver
// loop and kernel dispatch.  No CPU fallback: every step of the path is a kernel
// in kernels.cuh / gemm_tc.cuh.
#include <cuda_runtime.h>

#include <cmath>
#include <complex>
#include <cstdio>
#include <cstring>
#include <map>
#include <mutex>
#include <new>
#include <string>
#include <utility>
#include <vector>

#include "../../include/gmmnlse.h"
#include "gemm_h.cuh"
#include "gemm_tc.cuh"
#include "kernels.cuh"

namespace {

thread_local std::string g_cuda_err;

#define GM_CUDA(call)                                                                     \
  do {                                                                                    \
    cudaError_t e_ = (call);                                                              \
    if (e_ != cudaSuccess) {                                                              \
      g_cuda_err = std::string(#call) + ": " + cudaGetErrorString(e_);                    \
      return GMMNLSE_ECUDA;                                                               \
    }                                                                                     \
  } while (0)

#define GM_TRY(call)                 \
  do {                               \
    int s_ = (call);                 \
    if (s_ < 0) return s_;           \
  } while (0)

using cd = std::complex<double>;

void host_fft(std::vector<cd>& a, int sign) {   // iterative radix-2, fp64; plan-time only
  const size_t n = a.size();
  for (size_t i = 1, j = 0; i < n; ++i) {
    size_t bit = n >> 1;
    for (; j & bit; bit >>= 1) j ^= bit;
    j ^= bit;
    if (i < j) std::swap(a[i], a[j]);
  }
  for (size_t len = 2; len <= n; len <<= 1) {
    const double ang = sign * 2.0 * M_PI / (double)len;
    for (size_t i = 0; i < n; i += len)
      for (size_t k = 0; k < len / 2; ++k) {
        const cd w(std::cos(ang * (double)k), std::sin(ang * (double)k));
        const cd u = a[i + k], v = a[i + k + len / 2] * w;
        a[i + k] = u + v;
        a[i + k + len / 2] = u - v;
      }
  }
}

// fp32 value rounded to TF32 (10 explicit mantissa bits), round to nearest even; finite inputs only
float round_tf32(double x) {
  float f = (float)x;
  uint32_t u;
  std::memcpy(&u, &f, 4);
  u += 0xFFFu + ((u >> 13) & 1u);
  u &= 0xFFFFE000u;
  std::memcpy(&f, &u, 4);
  return f;
}

typedef CUresult (*EncodeTiledFn)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*,
                                  const cuuint64_t*, const cuuint32_t*, const cuuint32_t*, CUtensorMapInterleave,
                                  CUtensorMapSwizzle, CUtensorMapL2promotion, CUtensorMapFloatOOBfill);

// fp32 tensor map, 128-byte swizzle span (16- or 32-byte atoms); dims/box innermost first; strides in bytes for dims 1..rank-1
int encode_tmap(CUtensorMap* out, CUtensorMapDataType dtype, void* base, int rank, const cuuint64_t* dims,
                const cuuint64_t* strides, const cuuint32_t* box, CUtensorMapSwizzle swz) {
  static EncodeTiledFn fn = nullptr;
  if (!fn) {
    void* ptr = nullptr;
    cudaDriverEntryPointQueryResult q;
    cudaError_t e = cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &ptr, cudaEnableDefault, &q);
    if (e != cudaSuccess || q != cudaDriverEntryPointSuccess || !ptr) {
      g_cuda_err = "cudaGetDriverEntryPoint(cuTensorMapEncodeTiled) failed";
      return GMMNLSE_ECUDA;
    }
    fn = (EncodeTiledFn)ptr;
  }
  const cuuint32_t estr[5] = {1, 1, 1, 1, 1};
  CUresult r = fn(out, dtype, (cuuint32_t)rank, base, dims, strides, box, estr,
                  CU_TENSOR_MAP_INTERLEAVE_NONE, swz, CU_TENSOR_MAP_L2_PROMOTION_L2_256B,
                  CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
  if (r != CUDA_SUCCESS) {
    g_cuda_err = "cuTensorMapEncodeTiled failed with CUresult " + std::to_string((int)r);
    return GMMNLSE_ECUDA;
  }
  return 0;
}

int encode_tmap_f32(CUtensorMap* out, void* base, int rank, const cuuint64_t* dims, const cuuint64_t* strides,
                    const cuuint32_t* box, CUtensorMapSwizzle swz) {
  return encode_tmap(out, CU_TENSOR_MAP_DATA_TYPE_FLOAT32, base, rank, dims, strides, box, swz);
}

// cudaFuncAttributeMaxDynamicSharedMemorySize is a property of (device, kernel), not of the process: remember the
// largest size granted per pair and only ever raise it (plans on several devices, or of several shapes, share kernels).
std::mutex g_attr_mu;
std::map<std::pair<int, const void*>, size_t> g_attr;
int ensure_dyn_smem(int device, const void* fn, size_t bytes) {
  std::lock_guard<std::mutex> lk(g_attr_mu);
  size_t& have = g_attr[std::make_pair(device, fn)];
  if (bytes <= have || bytes <= 48 * 1024) return 0;
  GM_CUDA(cudaFuncSetAttribute(fn, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)bytes));
  have = bytes;
  return 0;
}

struct DeviceGuard {            // run a call on the plan's device, restore the caller's current device afterwards
  int prev = -1;
  bool switched = false;
  explicit DeviceGuard(int dev) {
    if (cudaGetDevice(&prev) == cudaSuccess && prev != dev) switched = cudaSetDevice(dev) == cudaSuccess;
  }
  ~DeviceGuard() {
    if (switched) cudaSetDevice(prev);
  }
};

int ilog2(int n) {
  int l = 0;
  while ((1 << l) < n) ++l;
  return l;
}

}  // namespace

// ============================================================================================
struct gmmnlse_plan {
  int P = 0, N = 0, M = 0, log2N = 0, Q = 0, precision = 0, shock = 1, max_iter = 0, fixed_iter = 0;
  int contraction = 0, raman = 0, graph = 0, stop_rule = 0, async_call = 0;
  int loop_state = 0;                      // 0 host loop so far, 1 device loop (CUDA graph) in use, -1 graph build failed
  int device = 0;                          // the CUDA device the plan was created on (every call runs there)
  // general form of Eq. 1 (gmmnlse_plan_create_general): separate, possibly complex tensors, no symmetry
  bool general = false, gen_complex = false;
  const double* gen_SR = nullptr;          // host, valid during init only
  double dt = 0, dz = 0, f_R = 0, omega0 = 0, n2 = 0, tol = 1e-6;
  cudaStream_t stream = nullptr;
  long long n_large = 0, n_iter = 0, n_noconv = 0, n_launch = 0;
  double last_err = 0;
  std::vector<double> phi;   // Im D_w^(p) [P][N]
  // per-kernel-class CUDA-event timing (gmmnlse_profile_*): event pairs recorded on `stream`
  bool prof_on = false;
  std::vector<cudaEvent_t> prof_ev;
  std::vector<int> prof_kind;
  size_t prof_used = 0;
  double prof_ms[GMMNLSE_KIND_COUNT] = {0};
  long long prof_n[GMMNLSE_KIND_COUNT] = {0};
  void prof_begin(int kind) {
    ++n_launch;
    if (!prof_on) return;
    if (prof_used + 2 > prof_ev.size()) {
      const size_t old = prof_ev.size();
      prof_ev.resize(old + 1024);
      for (size_t i = old; i < prof_ev.size(); ++i) cudaEventCreate(&prof_ev[i]);
    }
    prof_kind.push_back(kind);
    cudaEventRecord(prof_ev[prof_used++], stream);
  }
  void prof_end() {
    if (prof_on) cudaEventRecord(prof_ev[prof_used++], stream);
  }
  int prof_collect() {   // waits for the recorded events
    // wait for the last recorded event, not for `stream`: a per-call stream argument is no longer bound to the plan
    if (prof_used > 0 && cudaEventSynchronize(prof_ev[prof_used - 1]) != cudaSuccess) return GMMNLSE_ECUDA;
    for (size_t i = 0; i + 1 < prof_used; i += 2) {
      float ms = 0;
      if (cudaEventElapsedTime(&ms, prof_ev[i], prof_ev[i + 1]) != cudaSuccess) return GMMNLSE_ECUDA;
      const int k = prof_kind[i / 2];
      prof_ms[k] += ms;
      ++prof_n[k];
    }
    prof_used = 0;
    prof_kind.clear();
    return 0;
  }
  virtual ~gmmnlse_plan() {
    for (auto e : prof_ev) cudaEventDestroy(e);
  }
  virtual int init(const double* S, const double* h_R) = 0;
  virtual int propagate(const void* A_in, double L, void* A_out) = 0;
  virtual int propagate_host(const void* A_in, double L, void* A_out) = 0;
  virtual int propagate_rk4ip(const void* A_in, double L, void* A_out) = 0;
  virtual int set_gain(const double* g) = 0;
  virtual int set_coupling(const double* Qri) = 0;
  virtual int set_coupling_profile(const double* f, int n) = 0;
  virtual int set_gain_saturation(double g) = 0;
  virtual int shard_begin(const void* A_in) = 0;
  virtual int shard_iterate(int j_lo, int j_hi, int Mc, int first, void* block_sum) = 0;
  virtual int shard_update(int j_lo, int j_hi, int Mc, int first, const void* all_sums, int shard, int n_shards,
                           double* err_local) = 0;
  virtual int shard_advance(int Mc, const void* all_sums, int n_shards) = 0;
  virtual int shard_end(void* A_out) = 0;
  virtual int nonlinear_op(const void* A, void* dA) = 0;
  virtual int get_planes(void* out) = 0;
  virtual int debug_fft(const void* in, void* out, int rows, int dir) = 0;
  virtual int debug_pairs(const void* A, void* V, int n_planes) = 0;
  virtual int debug_contract(const void* V, void* U, int n_planes) = 0;
  virtual int contraction_kind() const = 0;
  virtual int set_tc_chunk(int k) = 0;
  virtual int raman_kind() const = 0;
  virtual int lowrank_rank() const = 0;
  virtual int sparse_info(int* classes, double* work_fraction) const = 0;
  virtual void drop_loop_graph() = 0;
  virtual int fold_pending() = 0;          // async calls: wait for the last call and take its loop counters in
};

namespace {

using namespace gm;

template <typename T>
struct PlanT final : gmmnlse_plan {
  using C = cplx<T>;
  // device tables
  C *tw = nullptr, *Kw = nullptr, *H = nullptr, *E = nullptr;
  double2* EM_d = nullptr;
  T* S2 = nullptr;
  int *pair_m = nullptr, *pair_n = nullptr;
  // device state
  double2* psi0_d = nullptr;
  C *psi = nullptr, *At = nullptr, *G = nullptr;   // [(M+1)][P][N]; psi plane 0 is psi_0
  T *V = nullptr, *U = nullptr;                    // [(M+1)][Q][N]
  double *errbuf = nullptr, *d_err = nullptr, *h_err = nullptr;
  void *h_in = nullptr, *h_out = nullptr;          // pinned staging for propagate_host
  C* d_io = nullptr;
  void* d2h_dst = nullptr;                         // set by propagate_host around its propagate() call
  size_t d2h_bytes = 0;
  std::map<int, double2*> EM_ragged;
  // device-side MPA loop: one CUDA graph per full large step = iteration 0, a WHILE node whose body is one further
  // iteration, a11.  k_err_finalize_loop takes the convergence decision; the host reads LoopStats once per call.
  cudaGraph_t lg = nullptr;
  cudaGraphExec_t lg_exec = nullptr;
  cudaStream_t cap_stream = nullptr;
  LoopStats *d_stats = nullptr, *h_stats = nullptr;
  long long lg_c0 = 0, lg_cb = 0, lg_ca = 0;       // kernel launches in iteration 0, the loop body, a11
  bool warmed = false;                             // one host-loop large step has run (function attributes set)
  // options.async_call: counters of the last call still on the device (copy to h_stats enqueued on pending_stream)
  long long pending_gsteps = 0;
  bool pending_last_on_device = false;
  cudaStream_t pending_stream = nullptr;
  void take_loop_stats(long long gsteps, bool last_on_device, int* status) {
    n_iter += h_stats->iters;
    n_launch += gsteps * (lg_c0 - lg_cb + lg_ca) + lg_cb * h_stats->iters;
    if (h_stats->noconv > 0) { n_noconv += h_stats->noconv; if (status) *status = GMMNLSE_WARN_NOCONV; }
    if (last_on_device) last_err = h_stats->last_err;
  }
  int fold_pending() override {
    if (pending_gsteps == 0) return 0;
    GM_CUDA(cudaStreamSynchronize(pending_stream));
    take_loop_stats(pending_gsteps, pending_last_on_device, nullptr);
    pending_gsteps = 0;
    return 0;
  }
  // serial RK4IP: one step (4 stages) as a graph, replayed; no decision inside, so no conditional node
  cudaGraph_t rkg = nullptr;
  cudaGraphExec_t rkg_exec = nullptr;
  long long rk_c = 0;                              // kernel launches per RK4IP step
  bool rk_warmed = false, rk_graph_failed = false;
  long long PN = 0, QN = 0;
  // NEXT-3: small-signal gain g_p (joins D as its real part) and constant linear coupling Q_np
  std::vector<double> gain;                // [P], 1/m; empty = none
  T *gfwd = nullptr, *ginv = nullptr;      // [(M+1)][P]: exp(+g_p j dz), exp(-g_p j dz)
  C* Qc = nullptr;                         // [P][P], Qc[n P + p] = Q_np
  C* Xconst = nullptr;                     // [P][P] i Q: the extra-term matrix when it is the same for every plane
  C* Xext = nullptr;                       // [(M+1)][P][P] per-plane matrix i f(z_j) Q - g_sat W_j (k_ext_matrix)
  T* Epair = nullptr;                      // [(M+1)][Q] time-integrated pair products (gain saturation)
  double g_sat = 0;                        // first-order gain saturation coefficient g0 / I_sat [m/J], 0 = off
  double* fprof_d = nullptr;               // z-profile of the coupling, sampled every dz / 2 from the start of a call
  int n_fprof = 0;
  int* d_step2 = nullptr;                  // device: twice the small steps taken so far in the current call
  int Bp = 0;                              // general mode: rows per Re / Im block of U, streams per Kerr / Raman block
  int* st_kind = nullptr;
  T *st_wk = nullptr, *st_wr = nullptr;
  StreamSpec<T> spec() const { return StreamSpec<T>{st_kind, st_wk, st_wr}; }
  // recursive Raman path (k_pair_iir): h_R[j] = Im(c zeta^j) detected from the samples
  bool iir = false;
  C iir_zeta, iir_cs, *iir_zp = nullptr;
  T iir_omf = 0;
  // register-blocked form of the recurrence (k_pair_iir_rows): complex64 scalar-mode plans with 512 <= N <= 8192
  // whose response has decayed to < 1e-12 over one warp's 512 samples
  bool iir_rows = false;
  PairWork* pair_work = nullptr;
  int n_pair_work = 0;
  ZetaPow iir_zk;
  std::map<const void*, CUtensorMap> field_tmaps;   // field buffer -> TMA map (the plan's At, or a caller's array)
  // serial RK4IP comparison integrator (allocated on first use)
  C *rk_X = nullptr, *rk_AI = nullptr, *rk_K1 = nullptr, *rk_K2 = nullptr, *rk_K3 = nullptr;
  double2* EH_d = nullptr;
  // tcgen05 contraction (complex64 path only): TF32 hi/lo split of S2, zero-padded to [R_pad][Q_pad]
  float *S2hi = nullptr, *S2lo = nullptr;
  CUtensorMap tmV, tmShi, tmSlo;
  // NEXT-4: exact low-rank form of the contraction, S_(pl),(mn) = sum_k L_(pl),k L_(mn),k (pivoted Cholesky)
  struct TcGemm {              // one rows x K operand of the single-CTA shared-memory tcgen05 kernel
    float *hi = nullptr, *lo = nullptr;
    CUtensorMap tmHi, tmLo;
    int rows = 0, K = 0, NT = 0, nrt = 0, KB = 0, stages = 0;
  };
  bool lowrank = false;
  int lr_R = 0;
  TcGemm lr1, lr2;             // Z = (L^T D) V  [R x Q],  U = L Z  [Q x R]
  T* Zb = nullptr;             // [(M+1)][R][N]
  CUtensorMap tmZ;
  // kind::f16 forms (gemm_h.cuh; options 7 dense, 8 low-rank): fp16 hi/lo split of both operands
  struct HGemm {
    __half *hi = nullptr, *lo = nullptr;
    float* rscale = nullptr;   // [nrt * NT] 1 / sS[r]
    CUtensorMap tmHi, tmLo;
    int rows = 0, K = 0, NT = 0, nrt = 0, KB = 0, stages = 0;
    double gain = 0;           // max_r sum_q |mat[r][q]|: |out| <= gain max |in|
  };
  bool tc_h = false;
  HGemm hg, hl1, hl2;
  // block-sparse form (options.contraction = 9): classes of packed pairs that S2 does not couple
  bool sparse = false;
  int sp_classes = 0, sp_Qv = 0;             // number of classes; rows of the class-ordered, padded V planes
  int *sp_kb_begin = nullptr, *sp_kb_count = nullptr, *sp_rowmap = nullptr, *sp_vrow = nullptr;
  T* Vsp = nullptr;                          // [(M+1)][sp_Qv][N] (as fp16 hi rows then lo rows per plane)
  double sp_work_fraction = 1.0;             // executed / dense multiply-adds
  float* d_vbound = nullptr;   // device scalar: bound on |V| of the current launch
  float v_gain = 1.f;          // |V| <= v_gain max |A|^2
  HalfOut cur_ho = {nullptr, 0, 0, 0, nullptr};
  CUtensorMap tmVh, tmVl, tmZh, tmZl;
  bool tc_on = false;          // dense 3xTF32 form (gemm_tc.cuh)
  int tc_NT = 0, tc_nrt = 0, tc_KB = 0, tc_stages = 0, tc_kchunk = 4, n_sm = 0;
  template <typename F> int ensure_smem(F fn, size_t bytes) { return ensure_dyn_smem(device, (const void*)fn, bytes); }
  // Every kernel goes out with programmatic stream serialisation (PDL): the next kernel on the stream may be
  // scheduled while this one drains and blocks in pdl_wait() until it has completed.  Captured into the loop graphs
  // this turns the kernel-to-kernel edges into programmatic ones (the launch-bound small configurations).
  bool pdl = true;
  cudaLaunchAttribute pdl_attr[1];
  void pdl_config(cudaLaunchConfig_t& cfg) {
    pdl_attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    pdl_attr[0].val.programmaticStreamSerializationAllowed = 1;
    cfg.attrs = pdl_attr;
    cfg.numAttrs = pdl ? 1 : 0;
  }
  template <typename... KArgs, typename... Args>
  void launch_k(void (*kern)(KArgs...), dim3 grid, dim3 block, size_t smem, Args&&... args) {
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = grid;
    cfg.blockDim = block;
    cfg.dynamicSmemBytes = smem;
    cfg.stream = stream;
    pdl_config(cfg);
    cudaLaunchKernelEx(&cfg, kern, static_cast<KArgs>(std::forward<Args>(args))...);   // errors: cudaGetLastError() at the call site
  }

  ~PlanT() override {
    cudaFree(tw); cudaFree(Kw); cudaFree(H); cudaFree(E); cudaFree(EM_d); cudaFree(S2);
    cudaFree(pair_m); cudaFree(pair_n); cudaFree(psi0_d); cudaFree(psi); cudaFree(At); cudaFree(G);
    cudaFree(V); cudaFree(U); cudaFree(errbuf); cudaFree(d_err); cudaFree(d_io);
    cudaFree(S2hi); cudaFree(S2lo);
    cudaFree(lr1.hi); cudaFree(lr1.lo); cudaFree(lr2.hi); cudaFree(lr2.lo); cudaFree(Zb);
    for (HGemm* g : {&hg, &hl1, &hl2}) { cudaFree(g->hi); cudaFree(g->lo); cudaFree(g->rscale); }
    cudaFree(d_vbound);
    drop_loop_graph();
    if (cap_stream) cudaStreamDestroy(cap_stream);
    cudaFree(d_stats);
    if (h_stats) cudaFreeHost(h_stats);
    cudaFree(gfwd); cudaFree(ginv); cudaFree(Qc); cudaFree(Xconst); cudaFree(Xext); cudaFree(Epair); cudaFree(fprof_d); cudaFree(d_step2); cudaFree(shard_pre);
    cudaFree(sp_kb_begin); cudaFree(sp_kb_count); cudaFree(sp_rowmap); cudaFree(sp_vrow); cudaFree(Vsp); cudaFree(st_kind); cudaFree(st_wk); cudaFree(st_wr); cudaFree(iir_zp); cudaFree(pair_work); cudaFree(rk_X); cudaFree(rk_AI); cudaFree(rk_K1); cudaFree(rk_K2); cudaFree(rk_K3); cudaFree(EH_d);
    if (h_err) cudaFreeHost(h_err);
    if (h_in) cudaFreeHost(h_in);
    if (h_out) cudaFreeHost(h_out);
    for (auto& kv : EM_ragged) cudaFree(kv.second);
  }

  template <typename X> int dalloc(X** p, size_t n) {
    cudaError_t e = cudaMalloc((void**)p, n * sizeof(X));
    if (e == cudaErrorMemoryAllocation) { cudaGetLastError(); return GMMNLSE_ENOMEM; }
    GM_CUDA(e);
    return 0;
  }
  template <typename X> int upload(X* d, const std::vector<X>& h) {
    GM_CUDA(cudaMemcpy(d, h.data(), h.size() * sizeof(X), cudaMemcpyHostToDevice));
    return 0;
  }

  int make_EM(int Mc, double2** out) {
    std::vector<double2> em((size_t)PN);
    for (long long i = 0; i < PN; ++i) {
      const double ph = std::remainder(phi[i] * (Mc * dz), 2.0 * M_PI);
      const double mag = gain.empty() ? 1.0 : std::exp(gain[(size_t)(i / N)] * (Mc * dz));
      em[i] = make_double2(mag * std::cos(ph), mag * std::sin(ph));
    }
    GM_TRY(dalloc(out, (size_t)PN));
    return upload(*out, em);
  }

  int init(const double* S, const double* h_R) override {
    PN = (long long)P * N;
    const int Qs = P * (P + 1) / 2;                  // unordered pairs m <= n
    Bp = (P * P + 1) & ~1;                           // P^2 rounded up to even
    Q = general ? 2 * Bp : Qs;
    QN = (long long)Q * N;
    // ---- tables (fp64 on the host, rounded once to T) ----
    std::vector<double> omega(N);
    for (int k = 0; k < N; ++k) omega[k] = 2.0 * M_PI * (double)(k < N / 2 ? k : k - N) / (N * dt);
    std::vector<C> h_tw(N), h_K(N), h_H(N);
    for (int m = 0; m < N; ++m) {
      const double a = 2.0 * M_PI * (double)m / (double)N;
      h_tw[m] = mk((T)std::cos(a), (T)std::sin(a));
    }
    const double kappa = n2 * omega0 / 299792458.0;
    for (int k = 0; k < N; ++k) h_K[k] = mk((T)0, (T)(kappa * (shock ? 1.0 + omega[k] / omega0 : 1.0)));
    {
      std::vector<cd> hh(N, cd(0, 0));
      if (f_R != 0.0) {
        double hsum = 0;
        for (int k = 0; k < N; ++k) { hh[k] = h_R[k]; hsum += std::fabs(h_R[k]); }
        host_fft(hh, +1);
        // |(1 - f_R) x + f_R dt (h_R (*) x)| <= v_gain max |x|: the range bound of the fp16 pair streams
        v_gain = (float)(1.0001 * ((1.0 - f_R) + f_R * dt * hsum));
      }
      for (int k = 0; k < N; ++k) {
        // scalar-mode path: the blended transfer function; general path: ht_R / N alone (weights per stream)
        const cd v = general ? dt * hh[k] / (double)N : ((1.0 - f_R) + f_R * dt * hh[k]) / (double)N;
        h_H[k] = mk((T)v.real(), (T)v.imag());
      }
    }
    GM_TRY(fit_raman(h_R));
    std::vector<C> h_E((size_t)(M + 1) * PN);
    for (int j = 0; j <= M; ++j)
      for (long long i = 0; i < PN; ++i) {
        const double ph = std::remainder(phi[i] * (j * dz), 2.0 * M_PI);
        h_E[(size_t)j * PN + i] = mk((T)std::cos(ph), (T)std::sin(ph));
      }
    // ---- packed coupling matrix: rows (p<=l), columns (m<=n), off-diagonal columns doubled ----
    std::vector<int> pm(Q, 0), pn(Q, 0);
    std::vector<T> h_S2((size_t)Q * Q);
    std::vector<double> h_S2d((size_t)Q * Q, 0.0);
    if (!general) {
      int q = 0;
      for (int m = 0; m < P; ++m)
        for (int n = m; n < P; ++n, ++q) { pm[q] = m; pn[q] = n; }
      for (int r = 0; r < Q; ++r)
        for (int qq = 0; qq < Q; ++qq) {
          const size_t idx = (((size_t)pm[r] * P + pn[r]) * P + pm[qq]) * P + pn[qq];
          h_S2d[(size_t)r * Q + qq] = S[idx] * (pm[qq] == pn[qq] ? 1.0 : 2.0);
        }
    } else {
      // General form.  Streams (columns), two blocks of Bp: [Kerr | Raman]; inside a block the Qs streams
      // X_mn = Re(A_m A_n*), m <= n, then the Qs - P streams Y_mn = Im(A_m A_n*), m < n (T_nm = conj T_mn).
      // Rows, two blocks of Bp: Re U_pl then Im U_pl, (p, l) ordered, row p P + l.  With s = S_plmn (complex):
      //   sum_mn s_mn T_mn = sum_{m<=n} alpha_mn X_mn + sum_{m<n} beta_mn Y_mn,
      //   alpha = s_mm (m = n) or s_mn + s_nm,  beta = i (s_mn - s_nm).
      std::vector<int> kind(Q, 0);
      std::vector<T> wk(Q, (T)0), wr(Q, (T)0);
      for (int b = 0; b < 2; ++b) {
        int q = b * Bp;
        for (int m = 0; m < P; ++m)
          for (int n = m; n < P; ++n, ++q) { pm[q] = m; pn[q] = n; kind[q] = 0; }
        for (int m = 0; m < P; ++m)
          for (int n = m + 1; n < P; ++n, ++q) { pm[q] = m; pn[q] = n; kind[q] = 1; }
        for (int qq = b * Bp; qq < (b + 1) * Bp; ++qq) {
          wk[qq] = b == 0 ? (T)(1.0 - f_R) : (T)0;
          wr[qq] = b == 0 ? (T)0 : (T)f_R;
        }
      }
      const int stride = gen_complex ? 2 : 1;
      auto tens = [&](const double* Sx, int p, int l, int m, int n) {
        const size_t idx = ((((size_t)p * P + l) * P + m) * P + n) * stride;
        return cd(Sx[idx], gen_complex ? Sx[idx + 1] : 0.0);
      };
      for (int b = 0; b < 2; ++b) {
        const double* Sx = b == 0 ? S : gen_SR;
        for (int p = 0; p < P; ++p)
          for (int l = 0; l < P; ++l) {
            const size_t rr = (size_t)p * P + l, ri = (size_t)Bp + rr;
            for (int q = b * Bp; q < b * Bp + P * P; ++q) {
              const int m = pm[q], n = pn[q];
              cd c;
              if (kind[q] == 0) c = m == n ? tens(Sx, p, l, m, m) : tens(Sx, p, l, m, n) + tens(Sx, p, l, n, m);
              else c = cd(0, 1) * (tens(Sx, p, l, m, n) - tens(Sx, p, l, n, m));
              h_S2d[rr * Q + q] = c.real();
              h_S2d[ri * Q + q] = c.imag();
            }
          }
      }
      GM_TRY(dalloc(&st_kind, Q)); GM_TRY(upload(st_kind, kind));
      GM_TRY(dalloc(&st_wk, Q)); GM_TRY(upload(st_wk, wk));
      GM_TRY(dalloc(&st_wr, Q)); GM_TRY(upload(st_wr, wr));
    }
    for (size_t i = 0; i < h_S2.size(); ++i) h_S2[i] = (T)h_S2d[i];
    GM_TRY(dalloc(&tw, N)); GM_TRY(upload(tw, h_tw));
    GM_TRY(dalloc(&Kw, N)); GM_TRY(upload(Kw, h_K));
    GM_TRY(dalloc(&H, N)); GM_TRY(upload(H, h_H));
    GM_TRY(dalloc(&E, (size_t)(M + 1) * PN)); GM_TRY(upload(E, h_E));
    GM_TRY(make_EM(M, &EM_d));
    GM_TRY(dalloc(&S2, (size_t)Q * Q)); GM_TRY(upload(S2, h_S2));
    GM_TRY(dalloc(&pair_m, Q)); GM_TRY(upload(pair_m, pm));
    GM_TRY(dalloc(&pair_n, Q)); GM_TRY(upload(pair_n, pn));
    GM_TRY(dalloc(&psi0_d, (size_t)PN));
    GM_TRY(dalloc(&psi, (size_t)(M + 1) * PN));
    GM_TRY(dalloc(&At, (size_t)(M + 1) * PN));
    GM_TRY(dalloc(&G, (size_t)(M + 1) * PN));
    GM_TRY(dalloc(&V, (size_t)(M + 1) * QN));
    GM_TRY(dalloc(&U, (size_t)(M + 1) * QN));
    GM_TRY(dalloc(&d_step2, 1));
    GM_CUDA(cudaMemset(d_step2, 0, sizeof(int)));
    GM_TRY(dalloc(&errbuf, (size_t)2 * (M + 2)));
    GM_TRY(dalloc(&d_err, 1));
    GM_CUDA(cudaMemset(errbuf, 0, sizeof(double) * 2 * (M + 2)));
    GM_CUDA(cudaMemset(psi, 0, sizeof(C) * (size_t)(M + 1) * PN));
    GM_CUDA(cudaMallocHost((void**)&h_err, sizeof(double)));
    GM_TRY(init_tc(h_S2d));
    return 0;
  }

  // ------------------------------------------------------------------ recursive Raman detection
  // Is h_R[j] = Im(c zeta^j) (a damped oscillation sampled at j dt)?  Fit the two-term recurrence
  // h[j+2] = a1 h[j+1] + a2 h[j] on the leading samples, take zeta from x^2 = a1 x + a2, c from h[0], h[1],
  // and accept only if every one of the N samples is reproduced to 1e-10 of the peak and zeta^N < 1e-14.
  // options.raman: 0 auto, 1 force the FFT path, 2 require the recursive path (EUNSUPPORTED if it does not fit).
  int fit_raman(const double* h) {
    iir = false;
    if (f_R == 0.0 || raman == 1 || N < 32) return raman == 2 && f_R != 0.0 ? GMMNLSE_EUNSUPPORTED : 0;
    const int nfit = std::min(N - 2, 96);
    long double s11 = 0, s12 = 0, s22 = 0, b1 = 0, b2 = 0, hmax = 0;
    for (int jn = 0; jn < N; ++jn) hmax = std::max(hmax, (long double)std::fabs(h[jn]));
    for (int jn = 0; jn < nfit; ++jn) {
      const long double u = h[jn + 1], v = h[jn], y = h[jn + 2];
      s11 += u * u; s12 += u * v; s22 += v * v; b1 += u * y; b2 += v * y;
    }
    const long double det = s11 * s22 - s12 * s12;
    bool ok = hmax > 0 && std::fabs((double)det) > 1e-24 * (double)(s11 * s22);
    double a1 = 0, a2 = 0;
    if (ok) {
      a1 = (double)((b1 * s22 - b2 * s12) / det);
      a2 = (double)((s11 * b2 - s12 * b1) / det);
      ok = a1 * a1 + 4.0 * a2 < 0.0;                        // complex pole pair
    }
    cd zeta, c;
    if (ok) {
      zeta = cd(0.5 * a1, std::sqrt(-a2 - 0.25 * a1 * a1));
      c = cd((h[1] - h[0] * zeta.real()) / zeta.imag(), h[0]);
      const double lnm = std::log(std::abs(zeta)), arg = std::arg(zeta);
      ok = lnm < 0.0 && lnm * N < std::log(1e-14);
      for (int jn = 0; ok && jn < N; ++jn) {
        const cd zj = std::exp(lnm * jn) * cd(std::cos(arg * jn), std::sin(arg * jn));
        if (std::fabs(h[jn] - (c * zj).imag()) > 1e-10 * (double)hmax) ok = false;
      }
    }
    if (!ok) return raman == 2 ? GMMNLSE_EUNSUPPORTED : 0;
    const int NT = N / 16;
    std::vector<C> zp((size_t)NT + 33);
    const double lnm = std::log(std::abs(zeta)), arg = std::arg(zeta);
    for (size_t m = 0; m < zp.size(); ++m) {
      const double mag = std::exp(lnm * 16.0 * (double)m), ph = std::remainder(arg * 16.0 * (double)m, 2.0 * M_PI);
      zp[m] = mk((T)(mag * std::cos(ph)), (T)(mag * std::sin(ph)));
    }
    GM_TRY(dalloc(&iir_zp, zp.size()));
    GM_TRY(upload(iir_zp, zp));
    iir_zeta = mk((T)zeta.real(), (T)zeta.imag());
    const cd csd = general ? c * dt : c * (dt * f_R);      // general mode: f_R sits in the per-stream weights
    iir_cs = mk((T)csd.real(), (T)csd.imag());
    iir_omf = (T)(1.0 - f_R);
    iir = true;
    if (sizeof(T) == 4 && !general && log2N >= 9 && log2N <= 14 && lnm * 512.0 < std::log(1e-12)) {
      // work list: CTA = rows (m0, m0 + 1) against up to G rows n >= m0.  G = 8 amortises the two parked rows;
      // with few modes that leaves most SMs without a CTA, so G shrinks until a launch of M planes has two per SM
      int dev = 0, sms = 148;
      GM_CUDA(cudaGetDevice(&dev));
      GM_CUDA(cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev));
      int G = 8;
      auto n_ctas = [&](int g) { long long c = 0; for (int m0 = 0; m0 < P; m0 += 2) c += (P - m0 + g - 1) / g; return c * M; };
      while (G > 1 && n_ctas(G) < 2LL * sms) G /= 2;
      std::vector<PairWork> wl;
      for (int m0 = 0; m0 < P; m0 += 2)
        for (int nb = m0; nb < P; nb += G) wl.push_back(PairWork{m0, nb, std::min(P, nb + G)});
      for (int k = 0; k < 16; ++k) {
        const double mag = std::exp(lnm * k), ph = arg * k;
        iir_zk.re[k] = (float)(mag * std::cos(ph));
        iir_zk.im[k] = (float)(mag * std::sin(ph));
      }
      n_pair_work = (int)wl.size();
      GM_TRY(dalloc(&pair_work, wl.size()));
      GM_TRY(upload(pair_work, wl));
      iir_rows = true;
    }
    return 0;
  }

  template <int LOG2N>
  int launch_pairs_iir_t(const C* A, long long a_ps, T* Vout, long long v_ps, int planes) {
    constexpr int NT = (1 << LOG2N) / 16, NW = (NT + 31) / 32;
    const size_t smem = sizeof(C) * (fft_smem_elems(1 << LOG2N) + 2 * NW + 2);
    GM_TRY(general ? ensure_smem(k_pair_iir<T, LOG2N, true>, smem) : ensure_smem(k_pair_iir<T, LOG2N, false>, smem));
    prof_begin(GMMNLSE_KIND_PAIR_CONV);
    const dim3 grid((Q + 1) / 2, planes);
    if (general)
      launch_k(k_pair_iir<T, LOG2N, true>, grid, NT, smem, A, a_ps, Vout, v_ps, pair_m, pair_n, Q, iir_zeta, iir_cs,
                                                             iir_omf, iir_zp, spec(), cur_ho);
    else
      launch_k(k_pair_iir<T, LOG2N, false>, grid, NT, smem, A, a_ps, Vout, v_ps, pair_m, pair_n, Q, iir_zeta,
                                                              iir_cs, iir_omf, iir_zp, spec(), cur_ho);
    prof_end();
    GM_CUDA(cudaGetLastError());
    return 0;
  }
  // TMA map over a field buffer [planes][P][N] complex64 seen as [planes][P][N/16][32 floats]: one box = the 32 x
  // 128 B slice of a row that one warp of k_pair_iir_rows reads
  int field_tmap(const C* A, const CUtensorMap** out) {
    auto it = field_tmaps.find((const void*)A);
    if (it == field_tmaps.end()) {
      if (field_tmaps.size() > 64) field_tmaps.clear();
      CUtensorMap tm;
      const cuuint64_t dims[4] = {32, (cuuint64_t)N / 16, (cuuint64_t)P, (cuuint64_t)(M + 1)};
      const cuuint64_t strides[3] = {128, (cuuint64_t)N * 8, (cuuint64_t)PN * 8};
      const cuuint32_t box[4] = {32, 32, 1, 1};
      GM_TRY(encode_tmap_f32(&tm, (void*)A, 4, dims, strides, box, CU_TENSOR_MAP_SWIZZLE_128B));
      it = field_tmaps.emplace((const void*)A, tm).first;
    }
    *out = &it->second;
    return 0;
  }
  template <int LOG2N, int SEGS = 1>
  int launch_pairs_rows_t(const C* A, T* Vout, long long v_ps, int planes) {
    if constexpr (sizeof(T) != 4) {
      return GMMNLSE_EUNSUPPORTED;
    } else {
      constexpr int NW = (1 << LOG2N) / 512 / SEGS + (SEGS > 1 ? 1 : 0), NT = 32 * NW;   // + the halo warp
      const size_t smem = 1024 + (size_t)3 * NT * 128 + (size_t)2 * NW * 2 * sizeof(float2) + (size_t)NW * 16;
      const bool half = cur_ho.Vh != nullptr;
      // the map addresses whole planes from a base: the plan's own At (any plane offset) or a caller's array
      const bool own = A >= At && A < At + (size_t)(M + 1) * PN;
      const C* tbase = own ? At : A;
      const int plane0 = own ? (int)((A - At) / PN) : 0;
      if (plane0 + planes > M + 1) return GMMNLSE_EINVAL;
      const CUtensorMap* tm = nullptr;
      GM_TRY(field_tmap(tbase, &tm));
      GM_TRY(half ? ensure_smem(k_pair_iir_rows<LOG2N, true, SEGS>, smem)
                  : ensure_smem(k_pair_iir_rows<LOG2N, false, SEGS>, smem));
      prof_begin(GMMNLSE_KIND_PAIR_CONV);
      const dim3 grid(n_pair_work * SEGS, planes);
      if (half)
        launch_k(k_pair_iir_rows<LOG2N, true, SEGS>, grid, NT, smem, *tm, plane0, Vout, v_ps, P, pair_work, iir_zeta, iir_cs,
                                                                 iir_omf, iir_zp, cur_ho, iir_zk);
      else
        launch_k(k_pair_iir_rows<LOG2N, false, SEGS>, grid, NT, smem, *tm, plane0, Vout, v_ps, P, pair_work, iir_zeta, iir_cs,
                                                                  iir_omf, iir_zp, cur_ho, iir_zk);
      prof_end();
      GM_CUDA(cudaGetLastError());
      return 0;
    }
  }
  int launch_pairs_iir(const C* A, long long a_ps, T* Vout, long long v_ps, int planes) {
    if (iir_rows && (a_ps == PN || planes == 1)) {
      switch (log2N) {
        case 9: return launch_pairs_rows_t<9>(A, Vout, v_ps, planes);
        case 10: return launch_pairs_rows_t<10>(A, Vout, v_ps, planes);
        case 11: return launch_pairs_rows_t<11>(A, Vout, v_ps, planes);
        case 12: return launch_pairs_rows_t<12>(A, Vout, v_ps, planes);
        case 13: return launch_pairs_rows_t<13>(A, Vout, v_ps, planes);
        case 14: return launch_pairs_rows_t<14, 2>(A, Vout, v_ps, planes);     // two half-row segments + a halo warp
      }
    }
#define GM_IIR_CASE(L) case L: return launch_pairs_iir_t<L>(A, a_ps, Vout, v_ps, planes);
    switch (log2N) {
      GM_IIR_CASE(5) GM_IIR_CASE(6) GM_IIR_CASE(7) GM_IIR_CASE(8) GM_IIR_CASE(9) GM_IIR_CASE(10) GM_IIR_CASE(11)
      GM_IIR_CASE(12) GM_IIR_CASE(13)
      case 14:
        if constexpr (sizeof(T) == 4) return launch_pairs_iir_t<14>(A, a_ps, Vout, v_ps, planes);
        return GMMNLSE_EUNSUPPORTED;
    }
#undef GM_IIR_CASE
    return GMMNLSE_EUNSUPPORTED;
  }

  // ------------------------------------------------------------------ tcgen05 contraction setup
  // contraction option: 0 auto (tensor cores when Q >= 64), 1 CUDA cores, 2 tcgen05 cta_group::2,
  // 3 tcgen05 cta_group::1 with both operands in shared memory, 4 tcgen05 with V_hi/V_lo in tensor memory.
  int make_v_tmap(CUtensorMap* tm, const T* base, int planes) {
    const cuuint64_t dims[3] = {(cuuint64_t)N, (cuuint64_t)Q, (cuuint64_t)planes};
    const cuuint64_t strides[2] = {(cuuint64_t)N * 4, (cuuint64_t)QN * 4};
    const cuuint32_t box[3] = {32, tc::BK, 1};
    // t-contiguous operand: 32-byte swizzle atoms (the only MN-major layout kind::tf32 accepts)
    return encode_tmap_f32(tm, (void*)base, 3, dims, strides, box, CU_TENSOR_MAP_SWIZZLE_128B_ATOM_32B);
  }
  // A-operand map (shared-memory form) over [planes][Krows][N] streams
  int make_a_tmap(CUtensorMap* tm, const T* base, int Krows, int planes) {
    const cuuint64_t dims[3] = {(cuuint64_t)N, (cuuint64_t)Krows, (cuuint64_t)planes};
    const cuuint64_t strides[2] = {(cuuint64_t)N * 4, (cuuint64_t)Krows * N * 4};
    const cuuint32_t box[3] = {32, tc::BK, 1};
    return encode_tmap_f32(tm, (void*)base, 3, dims, strides, box, CU_TENSOR_MAP_SWIZZLE_128B_ATOM_32B);
  }
  int tc_build(TcGemm& g, const std::vector<double>& mat, int rows, int K, int smax) {
    g.rows = rows; g.K = K;
    g.nrt = (rows + 207) / 208;
    g.NT = (((rows + g.nrt - 1) / g.nrt) + 15) / 16 * 16;
    g.KB = (K + tc::BK - 1) / tc::BK;
    g.stages = tc::MAX_STAGES;
    while (g.stages > 1 && tc::smem_bytes(g.NT, g.stages) > (size_t)smax) --g.stages;
    const int Rp = g.nrt * g.NT, Kp = g.KB * tc::BK;
    std::vector<float> hi((size_t)Rp * Kp, 0.f), lo((size_t)Rp * Kp, 0.f);
    for (int r = 0; r < rows; ++r)
      for (int q = 0; q < K; ++q) {
        const double v = mat[(size_t)r * K + q];
        const float h = round_tf32(v);
        hi[(size_t)r * Kp + q] = h;
        lo[(size_t)r * Kp + q] = round_tf32(v - (double)h);
      }
    GM_TRY(dalloc(&g.hi, hi.size())); GM_TRY(upload(g.hi, hi));
    GM_TRY(dalloc(&g.lo, lo.size())); GM_TRY(upload(g.lo, lo));
    const cuuint64_t dims[2] = {(cuuint64_t)Kp, (cuuint64_t)Rp};
    const cuuint64_t strides[1] = {(cuuint64_t)Kp * 4};
    const cuuint32_t box[2] = {tc::BK, (cuuint32_t)g.NT};
    const CUtensorMapSwizzle bsw = tc::BK == 32 ? CU_TENSOR_MAP_SWIZZLE_128B : CU_TENSOR_MAP_SWIZZLE_64B;
    GM_TRY(encode_tmap_f32(&g.tmHi, g.hi, 2, dims, strides, box, bsw));
    return encode_tmap_f32(&g.tmLo, g.lo, 2, dims, strides, box, bsw);
  }
  int tc_run(const TcGemm& g, const CUtensorMap& amap, int plane0, T* out, long long out_ps, int planes) {
    if constexpr (sizeof(T) != 4) {
      return GMMNLSE_EUNSUPPORTED;
    } else {
      tc::Params prm = {};
      prm.U = out; prm.u_plane_stride = out_ps;
      prm.Q = g.rows; prm.N = N; prm.NT = g.NT; prm.KB = g.KB; prm.n_rt = g.nrt;
      prm.t_tiles = N / tc::TM;
      prm.total_tiles = planes * prm.t_tiles * g.nrt;
      prm.plane0 = plane0; prm.stages = g.stages; prm.kchunk = tc_kchunk;
      cudaLaunchConfig_t cfg = {};
      cfg.gridDim = dim3((unsigned)std::min(n_sm, prm.total_tiles));
      cfg.blockDim = dim3(tc::NTHREADS);
      cfg.dynamicSmemBytes = tc::smem_bytes(g.NT, g.stages);
      cfg.stream = stream;
      pdl_config(cfg);
      prof_begin(GMMNLSE_KIND_CONTRACT);
      cudaError_t e = cudaLaunchKernelEx(&cfg, tc::k_contract_tc, amap, g.tmHi, g.tmLo, prm);
      prof_end();
      GM_CUDA(e);
      return 0;
    }
  }
  // ------------------------------------------------------------------ kind::f16 form (gemm_h.cuh)
  int h_build(HGemm& g, const std::vector<double>& mat, int rows, int K, int smax, int force_NT = 0, bool allow_wide = false) {
    g.rows = rows; g.K = K;
    // NT <= 208 (three epilogue slices of <= 72 columns); the dense U-output form may use ONE tile of <= 240 (slices
    // of 80) when that covers all rows: the V tile is then loaded once instead of twice
    const int cap = allow_wide && rows > 208 && rows <= 240 ? 240 : 208;
    g.nrt = (rows + cap - 1) / cap;
    g.NT = (((rows + g.nrt - 1) / g.nrt) + 15) / 16 * 16;
    if (force_NT > 0) { g.NT = force_NT; g.nrt = (rows + force_NT - 1) / force_NT; }
    g.KB = (K + hc::BK - 1) / hc::BK;
    g.stages = hc::MAX_STAGES;
    while (g.stages > 1 && hc::smem_bytes(g.NT, g.stages) > (size_t)smax) --g.stages;
    // measured at config 5 (r02): 3 stages of 43 KB 0.807 ms per 20-plane launch, 5 stages 0.834 ms, 2 stages 1.018 ms
    if (g.stages * hc::stage_bytes(g.NT) > 3 * 43520) g.stages = std::max(3, (3 * 43520) / hc::stage_bytes(g.NT));
    if (hc::smem_bytes(g.NT, g.stages) > (size_t)smax) return GMMNLSE_EUNSUPPORTED;
    const int Rp = g.nrt * g.NT, Kp = g.KB * hc::BK;
    std::vector<__half> hi((size_t)Rp * Kp, __float2half_rn(0.f)), lo((size_t)Rp * Kp, __float2half_rn(0.f));
    std::vector<float> rs((size_t)Rp, 1.f);
    g.gain = 0;
    for (int r = 0; r < rows; ++r) {
      double amax = 0, asum = 0;
      for (int q = 0; q < K; ++q) {
        const double a = std::fabs(mat[(size_t)r * K + q]);
        amax = std::fmax(amax, a);
        asum += a;
      }
      g.gain = std::fmax(g.gain, asum);
      int e = 0;
      if (amax > 0) std::frexp(amax, &e);                       // amax = m 2^e, m in [0.5, 1): scaled row max in [2^13, 2^14)
      const int sh = amax > 0 ? std::max(-120, std::min(120, hc::V_RANGE_LOG2 - e)) : 0;
      rs[r] = (float)std::ldexp(1.0, -sh);
      for (int q = 0; q < K; ++q) {
        const double v = std::ldexp(mat[(size_t)r * K + q], sh);
        const __half h = __float2half_rn((float)v);
        hi[(size_t)r * Kp + q] = h;
        lo[(size_t)r * Kp + q] = __float2half_rn((float)(v - (double)__half2float(h)));
      }
    }
    g.gain *= 1.0001;
    GM_TRY(dalloc(&g.hi, hi.size())); GM_TRY(upload(g.hi, hi));
    GM_TRY(dalloc(&g.lo, lo.size())); GM_TRY(upload(g.lo, lo));
    GM_TRY(dalloc(&g.rscale, rs.size())); GM_TRY(upload(g.rscale, rs));
    const cuuint64_t dims[2] = {(cuuint64_t)Kp, (cuuint64_t)Rp};
    const cuuint64_t strides[1] = {(cuuint64_t)Kp * 2};
    const cuuint32_t box[2] = {hc::BK, (cuuint32_t)g.NT};
    GM_TRY(encode_tmap(&g.tmHi, CU_TENSOR_MAP_DATA_TYPE_FLOAT16, g.hi, 2, dims, strides, box, CU_TENSOR_MAP_SWIZZLE_64B));
    return encode_tmap(&g.tmLo, CU_TENSOR_MAP_DATA_TYPE_FLOAT16, g.lo, 2, dims, strides, box, CU_TENSOR_MAP_SWIZZLE_64B);
  }
  // A-operand maps over fp16 split planes: plane = [Krows][N] hi rows then [Krows][N] lo rows
  int h_a_tmaps(CUtensorMap* mhi, CUtensorMap* mlo, const void* base, int Krows, int planes) {
    const cuuint64_t dims[3] = {(cuuint64_t)N, (cuuint64_t)Krows, (cuuint64_t)planes};
    const cuuint64_t strides[2] = {(cuuint64_t)N * 2, (cuuint64_t)Krows * N * 4};
    const cuuint32_t box[3] = {64, hc::BK, 1};
    __half* b = reinterpret_cast<__half*>(const_cast<void*>(base));
    GM_TRY(encode_tmap(mhi, CU_TENSOR_MAP_DATA_TYPE_FLOAT16, b, 3, dims, strides, box, CU_TENSOR_MAP_SWIZZLE_128B));
    return encode_tmap(mlo, CU_TENSOR_MAP_DATA_TYPE_FLOAT16, b + (size_t)Krows * N, 3, dims, strides, box,
                       CU_TENSOR_MAP_SWIZZLE_128B);
  }
  int h_run(const HGemm& g, const CUtensorMap& mhi, const CUtensorMap& mlo, int plane0, T* outU, __half* outZ,
            long long out_ps, int planes, float bound_gain, float zgain) {
    if constexpr (sizeof(T) != 4) {
      return GMMNLSE_EUNSUPPORTED;
    } else {
      hc::Params prm = {};
      prm.U = outU; prm.Zh = outZ; prm.u_plane_stride = out_ps;
      prm.rscale = g.rscale; prm.vbound = d_vbound; prm.bound_gain = bound_gain; prm.zgain = zgain;
      prm.Q = g.rows; prm.N = N; prm.NT = g.NT; prm.KB = g.KB; prm.n_rt = g.nrt;
      prm.t_tiles = N / hc::TM;
      prm.total_tiles = planes * prm.t_tiles * g.nrt;
      prm.plane0 = plane0; prm.stages = g.stages;
      const bool sp = sparse && &g == &hg;
      if (sp) { prm.kb_begin = sp_kb_begin; prm.kb_count = sp_kb_count; prm.rowmap = sp_rowmap; }
      prm.kchunk = tc_kchunk;                                    // k-blocks of 32 q here (16 q in the TF32 forms)
      cudaLaunchConfig_t cfg = {};
      cfg.gridDim = dim3((unsigned)std::min(n_sm, prm.total_tiles));
      cfg.blockDim = dim3(hc::NTHREADS);
      cfg.dynamicSmemBytes = hc::smem_bytes(g.NT, g.stages);
      cfg.stream = stream;
      pdl_config(cfg);
      prof_begin(GMMNLSE_KIND_CONTRACT);
      // tiles wider than 208 columns (one r-tile for 208 < Q <= 240: config 4's Q = 210) need 80 columns per epilogue
      // warp; the default instantiation keeps 72 (80 costs the config-5 kernel a spill and 1 %)
      const bool wide = g.NT > 208;
      if (wide && (outZ || sp)) return GMMNLSE_EUNSUPPORTED;
      cudaError_t e = outZ ? cudaLaunchKernelEx(&cfg, hc::k_contract_h<true>, mhi, mlo, g.tmHi, g.tmLo, prm)
                      : sp ? cudaLaunchKernelEx(&cfg, hc::k_contract_h<false, true>, mhi, mlo, g.tmHi, g.tmLo, prm)
                    : wide ? cudaLaunchKernelEx(&cfg, hc::k_contract_h<false, false, hc::EPI_COLS_WIDE>, mhi, mlo, g.tmHi,
                                                g.tmLo, prm)
                           : cudaLaunchKernelEx(&cfg, hc::k_contract_h<false>, mhi, mlo, g.tmHi, g.tmLo, prm);
      prof_end();
      GM_CUDA(e);
      return 0;
    }
  }
  int init_h_common(int smax) {
    GM_TRY(dalloc(&d_vbound, 1));
    GM_CUDA(cudaMemset(d_vbound, 0, sizeof(float)));
    GM_TRY(h_a_tmaps(&tmVh, &tmVl, V, Q, M + 1));
    if constexpr (sizeof(T) == 4) {
      GM_TRY(ensure_smem(hc::k_contract_h<false>, (size_t)smax));
      GM_TRY(ensure_smem(hc::k_contract_h<false, false, hc::EPI_COLS_WIDE>, (size_t)smax));
      GM_TRY(ensure_smem(hc::k_contract_h<true>, (size_t)smax));
    }
    tc_h = true;
    return 0;
  }

  // Pivoted Cholesky of the (p<=l) x (m<=n) symmetric matrix Ms = S_plmn (Eq. 2 makes it a Gram matrix of the
  // pair functions F_p F_l, hence positive semi-definite and, for Hermite-Gauss modes, of rank << Q).  Exact to
  // fp64 rounding: stops when the largest remaining diagonal is < 1e-13 of the largest, then verifies
  // max |Ms - L L^T| <= 1e-11 max |Ms| (a tensor that is not PSD fails here: EUNSUPPORTED).
  int init_lowrank(const std::vector<double>& h_S2, int smax) {
    std::vector<double> dbl(Q);
    for (int q = 0, m = 0; m < P; ++m)
      for (int n = m; n < P; ++n, ++q) dbl[q] = m == n ? 1.0 : 2.0;
    std::vector<double> Ms((size_t)Q * Q);
    double amax = 0;
    for (int r = 0; r < Q; ++r)
      for (int q = 0; q < Q; ++q) {
        Ms[(size_t)r * Q + q] = h_S2[(size_t)r * Q + q] / dbl[q];
        amax = std::fmax(amax, std::fabs(Ms[(size_t)r * Q + q]));
      }
    std::vector<double> d(Q), L;                       // L column-major by factor: L[k * Q + r]
    double dmax0 = 0;
    for (int r = 0; r < Q; ++r) { d[r] = Ms[(size_t)r * Q + r]; dmax0 = std::fmax(dmax0, d[r]); }
    if (!(dmax0 > 0)) return GMMNLSE_EUNSUPPORTED;
    int R = 0;
    while (R < Q) {
      int piv = 0;
      for (int r = 1; r < Q; ++r) if (d[r] > d[piv]) piv = r;
      if (d[piv] <= 1e-13 * dmax0) break;
      L.resize((size_t)(R + 1) * Q);
      double* col = &L[(size_t)R * Q];
      const double inv = 1.0 / std::sqrt(d[piv]);
      for (int r = 0; r < Q; ++r) {
        double v = Ms[(size_t)r * Q + piv];
        for (int k = 0; k < R; ++k) v -= L[(size_t)k * Q + r] * L[(size_t)k * Q + piv];
        col[r] = v * inv;
      }
      for (int r = 0; r < Q; ++r) d[r] -= col[r] * col[r];
      ++R;
    }
    double res = 0;
    for (int r = 0; r < Q; ++r)
      for (int q = r; q < Q; ++q) {
        double v = Ms[(size_t)r * Q + q];
        for (int k = 0; k < R; ++k) v -= L[(size_t)k * Q + r] * L[(size_t)k * Q + q];
        res = std::fmax(res, std::fabs(v));
      }
    if (R == 0 || res > 1e-11 * amax) return GMMNLSE_EUNSUPPORTED;
    lr_R = R;
    std::vector<double> W1((size_t)R * Q), W2((size_t)Q * R);
    for (int k = 0; k < R; ++k)
      for (int q = 0; q < Q; ++q) {
        W1[(size_t)k * Q + q] = L[(size_t)k * Q + q] * dbl[q];     // (L^T D)[k][q]
        W2[(size_t)q * R + k] = L[(size_t)k * Q + q];              // L[q][k]
      }
    if (contraction == 8) {                            // both GEMMs on the kind::f16 kernel, Z kept as fp16 hi / lo
      GM_TRY(h_build(hl1, W1, R, Q, smax));
      GM_TRY(h_build(hl2, W2, Q, R, smax));
      GM_TRY(dalloc(&Zb, (size_t)(M + 1) * R * N));
      GM_TRY(h_a_tmaps(&tmZh, &tmZl, Zb, R, M + 1));
      GM_TRY(init_h_common(smax));
      lowrank = true;
      return 0;
    }
    GM_TRY(tc_build(lr1, W1, R, Q, smax));
    GM_TRY(tc_build(lr2, W2, Q, R, smax));
    GM_TRY(dalloc(&Zb, (size_t)(M + 1) * R * N));
    GM_TRY(make_a_tmap(&tmZ, Zb, R, M + 1));
    GM_TRY(make_a_tmap(&tmV, V, Q, M + 1));
    if constexpr (sizeof(T) == 4) GM_TRY(ensure_smem(tc::k_contract_tc, (size_t)smax));
    lowrank = true;
    return 0;
  }

  // Block-sparse form of the dense contraction: the packed pairs fall into classes that S2 never couples (for the
  // Hermite-Gauss modes of a GRIN fibre: the four parities of the pair function F_p F_l in x and y; Eq. 2's integrand
  // is odd otherwise).  Classes = connected components of the graph r ~ q <=> |S2[r][q]| > 1e-13 max|S2| (union-find).
  // The operand is rebuilt with rows and columns in class order, each class's rows padded to whole r-tiles and its
  // columns to whole k-blocks, so an r-tile multiplies only its own class's k-blocks; the result is the dense
  // product up to the dropped entries (< 1e-13 of the largest).  One class only: EUNSUPPORTED (nothing to skip).
  int init_sparse(const std::vector<double>& h_S2, int smax) {
    double amax = 0;
    for (double v : h_S2) amax = std::fmax(amax, std::fabs(v));
    const double thr = 1e-13 * amax;
    std::vector<int> parent(Q);
    for (int i = 0; i < Q; ++i) parent[i] = i;
    auto find = [&](int x) { while (parent[x] != x) { parent[x] = parent[parent[x]]; x = parent[x]; } return x; };
    for (int r = 0; r < Q; ++r)
      for (int q = 0; q < Q; ++q)
        if (std::fabs(h_S2[(size_t)r * Q + q]) > thr) { const int a = find(r), b = find(q); if (a != b) parent[a] = b; }
    std::map<int, std::vector<int>> comp;
    for (int i = 0; i < Q; ++i) comp[find(i)].push_back(i);
    if (comp.size() < 2) return GMMNLSE_EUNSUPPORTED;
    std::vector<std::vector<int>> cls;
    for (auto& kv : comp) cls.push_back(kv.second);
    sp_classes = (int)cls.size();
    // tile height: the multiple of 16 in [16, 208] with the least cost.  Every r-tile re-reads its class's V k-blocks
    // (16 KB each: the shared-memory traffic of 128 rows of S2) and pays a drain per chunk, so a tile costs about
    // (NT + 128) per k-block, not NT: small tiles lose (NT = 16 measured 1.5x SLOWER than the dense form).
    int best_NT = 208;
    double best = 1e300, best_work = 0;
    for (int nt = 16; nt <= 208; nt += 16) {
      double cost = 0, work = 0;
      for (auto& c : cls) {
        const double tiles = (double)((c.size() + nt - 1) / nt), kq = (double)((c.size() + hc::BK - 1) / hc::BK * hc::BK);
        cost += tiles * (nt + 128) * kq;
        work += tiles * nt * kq;
      }
      if (cost <= best) { best = cost; best_NT = nt; best_work = work; }
    }
    sp_work_fraction = best_work / ((double)Q * Q);
    int Rp = 0, Kp = 0;
    std::vector<int> kb0, kbn, rowmap, vrow(Q, 0);
    for (auto& c : cls) {
      const int tiles = ((int)c.size() + best_NT - 1) / best_NT, kblocks = ((int)c.size() + hc::BK - 1) / hc::BK;
      for (int t = 0; t < tiles; ++t) { kb0.push_back(Kp / hc::BK); kbn.push_back(kblocks); }
      for (int i = 0; i < tiles * best_NT; ++i) rowmap.push_back(i < (int)c.size() ? c[i] : -1);
      for (int i = 0; i < (int)c.size(); ++i) vrow[c[i]] = Kp + i;
      Rp += tiles * best_NT;
      Kp += kblocks * hc::BK;
    }
    sp_Qv = Kp;
    std::vector<double> mat((size_t)Rp * Kp, 0.0);
    for (int rr = 0; rr < Rp; ++rr) {
      if (rowmap[rr] < 0) continue;
      const double* src = &h_S2[(size_t)rowmap[rr] * Q];
      for (int q = 0; q < Q; ++q)
        if (std::fabs(src[q]) > thr) mat[(size_t)rr * Kp + vrow[q]] = src[q];
    }
    GM_TRY(h_build(hg, mat, Rp, Kp, smax, best_NT));
    GM_TRY(dalloc(&sp_kb_begin, kb0.size())); GM_TRY(upload(sp_kb_begin, kb0));
    GM_TRY(dalloc(&sp_kb_count, kbn.size())); GM_TRY(upload(sp_kb_count, kbn));
    GM_TRY(dalloc(&sp_rowmap, rowmap.size())); GM_TRY(upload(sp_rowmap, rowmap));
    GM_TRY(dalloc(&sp_vrow, vrow.size())); GM_TRY(upload(sp_vrow, vrow));
    GM_TRY(dalloc(&Vsp, (size_t)(M + 1) * sp_Qv * N));
    GM_CUDA(cudaMemset(Vsp, 0, sizeof(T) * (size_t)(M + 1) * sp_Qv * N));     // the padding rows stay zero for good
    GM_TRY(dalloc(&d_vbound, 1));
    GM_CUDA(cudaMemset(d_vbound, 0, sizeof(float)));
    GM_TRY(h_a_tmaps(&tmVh, &tmVl, Vsp, sp_Qv, M + 1));
    if constexpr (sizeof(T) == 4) {
      GM_TRY(ensure_smem(hc::k_contract_h<false, true>, (size_t)smax));
      GM_TRY(ensure_smem(hc::k_contract_h<false>, (size_t)smax));
    }
    tc_h = true;
    sparse = true;
    return 0;
  }

  int init_tc(const std::vector<double>& h_S2) {
    if constexpr (sizeof(T) != 4) {
      if (contraction >= 2) return GMMNLSE_EUNSUPPORTED;
      return 0;
    } else {
      const bool want = contraction >= 2 || (contraction == 0 && Q >= 64);
      if (!want) return 0;
      // auto: the kind::f16 form wherever the tensor path applies (Q >= 64).  Measured against the 3xTF32 form:
      // +55 % at config 5, +18 % at config 4, +2 % at config 3 (r02: 19.7k vs 19.3k z-steps/s; in r01 the bound kernel
      // and memset in front of the pair kernel still cost more than they saved there)
      if (contraction == 7 || (contraction == 0 && N % hc::TM == 0)) {   // dense, fp16 hi / lo operands
        if (N % hc::TM != 0) return GMMNLSE_EUNSUPPORTED;
        int dev0 = 0, smax0 = 0;
        GM_CUDA(cudaGetDevice(&dev0));
        GM_CUDA(cudaDeviceGetAttribute(&n_sm, cudaDevAttrMultiProcessorCount, dev0));
        GM_CUDA(cudaDeviceGetAttribute(&smax0, cudaDevAttrMaxSharedMemoryPerBlockOptin, dev0));
        GM_TRY(h_build(hg, h_S2, Q, Q, smax0, 0, true));
        return init_h_common(smax0);
      }
      if (contraction == 9) {                          // block-sparse form (NEXT-4), scalar-mode path only
        if (general || N % hc::TM != 0) return GMMNLSE_EUNSUPPORTED;
        int dev0 = 0, smax0 = 0;
        GM_CUDA(cudaGetDevice(&dev0));
        GM_CUDA(cudaDeviceGetAttribute(&n_sm, cudaDevAttrMultiProcessorCount, dev0));
        GM_CUDA(cudaDeviceGetAttribute(&smax0, cudaDevAttrMaxSharedMemoryPerBlockOptin, dev0));
        return init_sparse(h_S2, smax0);
      }
      if (contraction == 6 || contraction == 8) {      // exact low-rank form (NEXT-4), scalar-mode path only
        if (general || N % tc::TM != 0) return GMMNLSE_EUNSUPPORTED;
        int dev0 = 0, smax0 = 0;
        GM_CUDA(cudaGetDevice(&dev0));
        GM_CUDA(cudaDeviceGetAttribute(&n_sm, cudaDevAttrMultiProcessorCount, dev0));
        GM_CUDA(cudaDeviceGetAttribute(&smax0, cudaDevAttrMaxSharedMemoryPerBlockOptin, dev0));
        return init_lowrank(h_S2, smax0);
      }
      // dense 3xTF32 form: single CTA per tile, both operands in shared memory
      if (N % tc::TM != 0) {
        if (contraction >= 2) return GMMNLSE_EUNSUPPORTED;
        return 0;
      }
      int dev = 0;
      GM_CUDA(cudaGetDevice(&dev));
      GM_CUDA(cudaDeviceGetAttribute(&n_sm, cudaDevAttrMultiProcessorCount, dev));
      tc_nrt = (Q + 207) / 208;                                  // NT <= 208: 3 epilogue slices of <= 72
      tc_NT = (((Q + tc_nrt - 1) / tc_nrt) + 15) / 16 * 16;
      tc_KB = (Q + tc::BK - 1) / tc::BK;
      const int Rp = tc_nrt * tc_NT, Qp = tc_KB * tc::BK;
      int smax = 0;
      GM_CUDA(cudaDeviceGetAttribute(&smax, cudaDevAttrMaxSharedMemoryPerBlockOptin, dev));
      tc_stages = tc::MAX_STAGES;
      while (tc_stages > 1 && tc::smem_bytes(tc_NT, tc_stages) > (size_t)smax) --tc_stages;
      if (tc::smem_bytes(tc_NT, tc_stages) > (size_t)smax) return GMMNLSE_EUNSUPPORTED;
      std::vector<float> hi((size_t)Rp * Qp, 0.f), lo((size_t)Rp * Qp, 0.f);
      for (int r = 0; r < Q; ++r)
        for (int q = 0; q < Q; ++q) {
          const double s = h_S2[(size_t)r * Q + q];
          const float h = round_tf32(s);
          hi[(size_t)r * Qp + q] = h;
          lo[(size_t)r * Qp + q] = round_tf32(s - (double)h);
        }
      GM_TRY(dalloc(&S2hi, hi.size())); GM_TRY(upload(S2hi, hi));
      GM_TRY(dalloc(&S2lo, lo.size())); GM_TRY(upload(S2lo, lo));
      const cuuint64_t dims[2] = {(cuuint64_t)Qp, (cuuint64_t)Rp};
      const cuuint64_t strides[1] = {(cuuint64_t)Qp * 4};
      const cuuint32_t box[2] = {tc::BK, (cuuint32_t)tc_NT};
      const CUtensorMapSwizzle bsw = tc::BK == 32 ? CU_TENSOR_MAP_SWIZZLE_128B : CU_TENSOR_MAP_SWIZZLE_64B;
      GM_TRY(encode_tmap_f32(&tmShi, S2hi, 2, dims, strides, box, bsw));
      GM_TRY(encode_tmap_f32(&tmSlo, S2lo, 2, dims, strides, box, bsw));
      GM_TRY(make_v_tmap(&tmV, V, M + 1));
      GM_TRY(ensure_smem(tc::k_contract_tc, tc::smem_bytes(tc_NT, tc_stages)));
      tc_on = true;
      return 0;
    }
  }

  int launch_contract_tc(const CUtensorMap& vmap, int plane0, T* Uout, int planes) {
    if constexpr (sizeof(T) != 4) {
      return GMMNLSE_EUNSUPPORTED;
    } else {
      tc::Params prm = {};
      prm.U = Uout;
      prm.u_plane_stride = QN;
      prm.Q = Q; prm.N = N; prm.NT = tc_NT; prm.KB = tc_KB; prm.n_rt = tc_nrt;
      prm.t_tiles = N / tc::TM;
      prm.total_tiles = planes * prm.t_tiles * tc_nrt;
      prm.plane0 = plane0; prm.stages = tc_stages; prm.kchunk = tc_kchunk;
      cudaLaunchConfig_t cfg = {};
      cfg.gridDim = dim3((unsigned)std::min(n_sm, prm.total_tiles));
      cfg.blockDim = dim3(tc::NTHREADS);
      cfg.dynamicSmemBytes = tc::smem_bytes(tc_NT, tc_stages);
      cfg.stream = stream;
      pdl_config(cfg);
      prof_begin(GMMNLSE_KIND_CONTRACT);
      cudaError_t e = cudaLaunchKernelEx(&cfg, tc::k_contract_tc, vmap, tmShi, tmSlo, prm);
      prof_end();
      GM_CUDA(e);
      return 0;
    }
  }

  // ------------------------------------------------------------------ kernel launchers
  template <int LOG2N, int DIR>
  int launch_fft_t(const C* in, long long in_ps, C* out, long long out_ps, const C* pre, const C* post_vec,
                   const C* post_tab, long long tab_ps, T scale, int rows, int planes, const T* rscale, float* bound) {
    constexpr int NT = (1 << LOG2N) / 16;
    const size_t smem = sizeof(C) * fft_smem_elems(1 << LOG2N);
    GM_TRY(ensure_smem(k_fft_rows<T, LOG2N, DIR>, smem));
    prof_begin(DIR > 0 ? GMMNLSE_KIND_FFT_TO_FREQ : GMMNLSE_KIND_FFT_TO_TIME);
    launch_k(k_fft_rows<T, LOG2N, DIR>, dim3(rows, planes), NT, smem, in, in_ps, out, out_ps, pre, post_vec,
             post_tab, tab_ps, scale, tw, rscale, bound, v_gain);
    prof_end();
    GM_CUDA(cudaGetLastError());
    return 0;
  }
  // bound != nullptr: also accumulate v_gain max |out|^2 into it (zeroed by the caller): see launch_pairs
  int launch_fft(int dir, const C* in, long long in_ps, C* out, long long out_ps, const C* pre, const C* post_vec,
                 const C* post_tab, long long tab_ps, T scale, int rows, int planes, const T* rscale = nullptr,
                 float* bound = nullptr) {
#define GM_FFT_CASE(L)                                                                                       \
  case L:                                                                                                    \
    return dir > 0 ? launch_fft_t<L, +1>(in, in_ps, out, out_ps, pre, post_vec, post_tab, tab_ps, scale, rows, \
                                         planes, rscale, bound)                                              \
                   : launch_fft_t<L, -1>(in, in_ps, out, out_ps, pre, post_vec, post_tab, tab_ps, scale, rows, \
                                         planes, rscale, bound);
    switch (log2N) {
      GM_FFT_CASE(4) GM_FFT_CASE(5) GM_FFT_CASE(6) GM_FFT_CASE(7) GM_FFT_CASE(8) GM_FFT_CASE(9)
      GM_FFT_CASE(10) GM_FFT_CASE(11) GM_FFT_CASE(12) GM_FFT_CASE(13)
      case 14:
        if constexpr (sizeof(T) == 4) {
          return dir > 0 ? launch_fft_t<14, +1>(in, in_ps, out, out_ps, pre, post_vec, post_tab, tab_ps, scale,
                                                rows, planes, rscale, bound)
                         : launch_fft_t<14, -1>(in, in_ps, out, out_ps, pre, post_vec, post_tab, tab_ps, scale,
                                                rows, planes, rscale, bound);
        }
        return GMMNLSE_EUNSUPPORTED;
    }
#undef GM_FFT_CASE
    return GMMNLSE_EUNSUPPORTED;
  }

  template <int LOG2N, bool RAMAN>
  int launch_pairs_t(const C* A, long long a_ps, T* Vout, long long v_ps, int planes) {
    constexpr int NT = (1 << LOG2N) / 16;
    const size_t smem = RAMAN ? sizeof(C) * fft_smem_elems(1 << LOG2N) : 0;
    GM_TRY(ensure_smem(k_pair_conv<T, LOG2N, RAMAN>, smem));
    prof_begin(GMMNLSE_KIND_PAIR_CONV);
    launch_k(k_pair_conv<T, LOG2N, RAMAN>, dim3((Q + 1) / 2, planes), NT, smem, A, a_ps, Vout, v_ps, pair_m,
                                                                                  pair_n, Q, H, tw, spec(), cur_ho);
    prof_end();
    GM_CUDA(cudaGetLastError());
    return 0;
  }
  bool own_v(const T* p) const { return p >= V && p < V + (size_t)(M + 1) * QN; }
  bool bound_from_fft = false;   // d_vbound already holds the bound of the planes the next launch_pairs works on
  int launch_pairs(const C* A, long long a_ps, T* Vout, long long v_ps, int planes) {
    cur_ho.Vh = nullptr;
    if constexpr (sizeof(T) == 4) {
      if (tc_h && own_v(Vout)) {                    // the f16 contraction follows: V as fp16 hi / lo planes
        if (!bound_from_fft) {                      // (the MPA iteration gets the bound from its a3 FFT's stores)
          GM_CUDA(cudaMemsetAsync(d_vbound, 0, sizeof(float), stream));
          prof_begin(GMMNLSE_KIND_PAIR_CONV);
          launch_k(k_bound_field<T>, dim3(32, planes), 256, 0, A, a_ps, PN, v_gain, d_vbound);
          prof_end();
          GM_CUDA(cudaGetLastError());
        }
        bound_from_fft = false;
        if (sparse) {                               // class-ordered, padded rows in the plan's Vsp planes
          const long long vq = (long long)sp_Qv * N;
          cur_ho = HalfOut{reinterpret_cast<__half*>(Vsp + ((Vout - V) / QN) * vq), 2 * vq, vq, N, d_vbound, sp_vrow};
        } else {
          cur_ho = HalfOut{reinterpret_cast<__half*>(Vout), 2 * QN, QN, N, d_vbound};
        }
      }
    }
    return launch_pairs_impl(A, a_ps, Vout, v_ps, planes);
  }
  int launch_pairs_impl(const C* A, long long a_ps, T* Vout, long long v_ps, int planes) {
    if (iir) return launch_pairs_iir(A, a_ps, Vout, v_ps, planes);
    const bool raman = f_R != 0.0;
#define GM_PC_CASE(L)                                                               \
  case L:                                                                           \
    return raman ? launch_pairs_t<L, true>(A, a_ps, Vout, v_ps, planes)             \
                 : launch_pairs_t<L, false>(A, a_ps, Vout, v_ps, planes);
    switch (log2N) {
      GM_PC_CASE(4) GM_PC_CASE(5) GM_PC_CASE(6) GM_PC_CASE(7) GM_PC_CASE(8) GM_PC_CASE(9)
      GM_PC_CASE(10) GM_PC_CASE(11) GM_PC_CASE(12) GM_PC_CASE(13)
      case 14:
        if constexpr (sizeof(T) == 4) {
          return raman ? launch_pairs_t<14, true>(A, a_ps, Vout, v_ps, planes)
                       : launch_pairs_t<14, false>(A, a_ps, Vout, v_ps, planes);
        }
        return GMMNLSE_EUNSUPPORTED;
    }
#undef GM_PC_CASE
    return GMMNLSE_EUNSUPPORTED;
  }

  int launch_contract(const T* Vin, T* Uout, int planes) {
    if constexpr (sizeof(T) == 4) {
      if (tc_h) {
        if (planes > M + 1) return GMMNLSE_EINVAL;
        int plane0 = 0;
        if (own_v(Vin)) {
          plane0 = (int)((Vin - V) / QN);
        } else {                                    // caller's fp32 V: bound, split into the plan's V planes
          const long long total = (long long)planes * QN;
          GM_CUDA(cudaMemsetAsync(d_vbound, 0, sizeof(float), stream));
          prof_begin(GMMNLSE_KIND_CONTRACT);
          launch_k(k_bound_real<T>, 592, 256, 0, Vin, total, d_vbound);
          const long long vq = (long long)sp_Qv * N;
          launch_k(k_v_encode, 1184, 256, 0, Vin, QN, total,
                   sparse ? HalfOut{reinterpret_cast<__half*>(Vsp), 2 * vq, vq, N, d_vbound, sp_vrow}
                          : HalfOut{reinterpret_cast<__half*>(V), 2 * QN, QN, N, d_vbound});
          prof_end();
          GM_CUDA(cudaGetLastError());
        }
        if (lowrank) {
          GM_TRY(h_run(hl1, tmVh, tmVl, plane0, nullptr, reinterpret_cast<__half*>(Zb), 2LL * lr_R * N, planes, 1.f,
                       (float)hl1.gain));
          return h_run(hl2, tmZh, tmZl, 0, Uout, nullptr, QN, planes, (float)hl1.gain, 0.f);
        }
        return h_run(hg, tmVh, tmVl, plane0, Uout, nullptr, QN, planes, 1.f, 0.f);
      }
    }
    if (lowrank) {
      if (planes > M + 1) return GMMNLSE_EINVAL;
      if (Vin >= V && Vin < V + (size_t)(M + 1) * QN) {
        GM_TRY(tc_run(lr1, tmV, (int)((Vin - V) / QN), Zb, (long long)lr_R * N, planes));
      } else {
        CUtensorMap tmp;
        GM_TRY(make_a_tmap(&tmp, Vin, Q, planes));
        GM_TRY(tc_run(lr1, tmp, 0, Zb, (long long)lr_R * N, planes));
      }
      return tc_run(lr2, tmZ, 0, Uout, QN, planes);
    }
    if (tc_on) {
      if (Vin >= V && Vin < V + (size_t)(M + 1) * QN)              // the plan's own buffer
        return launch_contract_tc(tmV, (int)((Vin - V) / QN), Uout, planes);
      CUtensorMap tmp;
      GM_TRY(make_v_tmap(&tmp, Vin, planes));
      return launch_contract_tc(tmp, 0, Uout, planes);
    }
    prof_begin(GMMNLSE_KIND_CONTRACT);
    if (Q <= 32) {
      constexpr int BM = 32, BN = 128, BK = 8, TM = 4, TN = 4;
      dim3 grid((N + BN - 1) / BN, (Q + BM - 1) / BM, planes);
      launch_k(k_contract<T, BM, BN, BK, TM, TN>, grid, (BM / TM) * (BN / TN), 0, S2, Vin, QN, Uout, QN, Q, N);
    } else {
      constexpr int BM = 128, BN = 128, BK = 8, TM = 8, TN = 8;
      dim3 grid((N + BN - 1) / BN, (Q + BM - 1) / BM, planes);
      launch_k(k_contract<T, BM, BN, BK, TM, TN>, grid, (BM / TM) * (BN / TN), 0, S2, Vin, QN, Uout, QN, Q, N);
    }
    prof_end();
    GM_CUDA(cudaGetLastError());
    return 0;
  }

  // TMA maps for the streaming a7: U (the plan's own buffer) and the field buffer seen as rows of float pairs
  CUtensorMap tmU7, tmA7;
  bool a7_maps = false;
  // slice width: 16 samples when the slice is large anyway (Q >= 256: 64 B x Q >= 16 KB), else 64 (measured at
  // Q = 120 / 210 with 16: the per-slice barrier and TMA issue cost more than the second read of U they save)
  int a7_tw() const { return Q >= 256 ? 16 : 64; }
  int a7_nbox() const { return (Q + 255) / 256; }
  int a7_rows_box() const { return (((Q + a7_nbox() - 1) / a7_nbox()) + 1) & ~1; }   // even: 128-byte aligned TMA boxes
  size_t a7_smem() const {
    return (size_t)2 * ((size_t)a7_nbox() * a7_rows_box() * 4 * a7_tw() + (size_t)P * 8 * a7_tw()) + 16 + 128;
  }
  int a7_stream_setup() {
    if (a7_maps) return 0;
    {
      const cuuint64_t dims[3] = {(cuuint64_t)N, (cuuint64_t)Q, (cuuint64_t)(M + 1)};
      const cuuint64_t strides[2] = {(cuuint64_t)N * 4, (cuuint64_t)QN * 4};
      const cuuint32_t box[3] = {(cuuint32_t)a7_tw(), (cuuint32_t)a7_rows_box(), 1};
      GM_TRY(encode_tmap_f32(&tmU7, (void*)U, 3, dims, strides, box, CU_TENSOR_MAP_SWIZZLE_NONE));
    }
    {
      const cuuint64_t dims[3] = {(cuuint64_t)2 * N, (cuuint64_t)P, (cuuint64_t)(M + 1)};
      const cuuint64_t strides[2] = {(cuuint64_t)N * 8, (cuuint64_t)PN * 8};
      const cuuint32_t box[3] = {(cuuint32_t)(2 * a7_tw()), (cuuint32_t)P, 1};
      GM_TRY(encode_tmap_f32(&tmA7, (void*)At, 3, dims, strides, box, CU_TENSOR_MAP_SWIZZLE_NONE));
    }
    a7_maps = true;
    return 0;
  }
  // streaming a7 applies to the plan's own U and At planes of a complex64 scalar-mode plan with enough slices to
  // occupy the device and a slice pair that fits shared memory
  bool a7_streams(const T* Uin, const C* A, int planes) const {
    if (sizeof(T) != 4 || general || N % 64 != 0 || P > 256 || n_sm <= 0 || Q < 64) return false;
    if (!(Uin >= U && Uin < U + (size_t)(M + 1) * QN) || !(A >= At && A < At + (size_t)(M + 1) * PN)) return false;
    return a7_smem() <= 200 * 1024 && (long long)planes * (N / a7_tw()) >= 4LL * n_sm;
  }

  int launch_mode_reduce(const T* Uin, const C* A, C* Nout, int planes) {
    if constexpr (sizeof(T) == 4) {
      if (a7_streams(Uin, A, planes)) {
        GM_TRY(a7_stream_setup());
        const size_t smem = a7_smem();
        const int tw7 = a7_tw();
        GM_TRY(tw7 == 16 ? ensure_smem(k_mode_reduce_stream<16>, smem) : ensure_smem(k_mode_reduce_stream<64>, smem));
        const int n_slices = planes * (N / tw7);
        prof_begin(GMMNLSE_KIND_MODE_REDUCE);
        cudaLaunchConfig_t cfg = {};
        cfg.gridDim = dim3((unsigned)std::min(n_sm, n_slices));
        // one mode per thread where the block size allows (16-sample slices: up to P = 64; 64-sample: up to 16)
        cfg.blockDim = dim3((unsigned)tw7 * (unsigned)std::min(1024 / tw7, (P + 1) & ~1));
        cfg.dynamicSmemBytes = smem;
        cfg.stream = stream;
        pdl_config(cfg);
        cudaError_t e = tw7 == 16
            ? cudaLaunchKernelEx(&cfg, k_mode_reduce_stream<16>, tmU7, tmA7, (int)((Uin - U) / QN), (int)((A - At) / PN),
                                 (float2*)Nout, PN, P, Q, N, n_slices, a7_nbox(), a7_rows_box())
            : cudaLaunchKernelEx(&cfg, k_mode_reduce_stream<64>, tmU7, tmA7, (int)((Uin - U) / QN), (int)((A - At) / PN),
                                 (float2*)Nout, PN, P, Q, N, n_slices, a7_nbox(), a7_rows_box());
        prof_end();
        GM_CUDA(e);
        return 0;
      }
    }
    if (general) {
      const size_t smem = sizeof(C) * P * 128;
      GM_TRY(ensure_smem(k_mode_reduce_gen<T>, smem));
      const int Gg = P >= 12 ? 4 : (P >= 4 ? 2 : 1);
      prof_begin(GMMNLSE_KIND_MODE_REDUCE);
      launch_k(k_mode_reduce_gen<T>, dim3((N + 127) / 128, planes), 128 * Gg, smem, Uin, QN, A, PN, Nout, PN, P, Bp,
                                                                                        N);
      prof_end();
      GM_CUDA(cudaGetLastError());
      return 0;
    }
    const int tw = P >= 32 && N >= 64 ? 32 : 128;                   // samples per CTA
    const int G = tw == 128 ? (P >= 12 ? 4 : (P >= 4 ? 2 : 1)) : 8; // mode groups per CTA
    const size_t smem = sizeof(C) * P * tw;
    GM_TRY(tw == 32 ? ensure_smem(k_mode_reduce<T, 32>, smem) : ensure_smem(k_mode_reduce<T, 128>, smem));
    const dim3 grid((N + tw - 1) / tw, planes);
    prof_begin(GMMNLSE_KIND_MODE_REDUCE);
    if (tw == 32) launch_k(k_mode_reduce<T, 32>, grid, 32 * G, smem, Uin, QN, A, PN, Nout, PN, P, N);
    else launch_k(k_mode_reduce<T, 128>, grid, 128 * G, smem, Uin, QN, A, PN, Nout, PN, P, N);
    prof_end();
    GM_CUDA(cudaGetLastError());
    return 0;
  }

  // small P (CUDA-core contraction, Q < 64, scalar-mode path): a6 + a7 -- and a4 when there is no Raman term -- in
  // one pointwise kernel, k_small_contract_reduce
  bool small_fused() const { return !general && !tc_h && !tc_on && !lowrank && P <= 10; }
  template <int PMAX, int SPLIT>
  int launch_small_t(const T* Vin, const C* A, C* Nout, int planes) {
    constexpr int TW = kSmallThreads / SPLIT, QMAX = PMAX * (PMAX + 1) / 2, KQ = (QMAX + SPLIT - 1) / SPLIT,
                  QP = (KQ * SPLIT + 3) & ~3;
    const bool inline_pairs = f_R == 0.0;
    const size_t smem = sizeof(T) * (size_t)QMAX * QP + sizeof(C) * (size_t)P * TW;
    GM_TRY(inline_pairs ? ensure_smem(k_small_contract_reduce<T, PMAX, SPLIT, true>, smem)
                        : ensure_smem(k_small_contract_reduce<T, PMAX, SPLIT, false>, smem));
    const dim3 grid((N + TW - 1) / TW, planes);
    prof_begin(GMMNLSE_KIND_CONTRACT);
    if (inline_pairs)
      launch_k(k_small_contract_reduce<T, PMAX, SPLIT, true>, grid, kSmallThreads, smem, S2, Vin, QN, A, PN, Nout, PN, pair_m,
                                                                                 pair_n, P, Q, N);
    else
      launch_k(k_small_contract_reduce<T, PMAX, SPLIT, false>, grid, kSmallThreads, smem, S2, Vin, QN, A, PN, Nout, PN, pair_m,
                                                                                  pair_n, P, Q, N);
    prof_end();
    GM_CUDA(cudaGetLastError());
    return 0;
  }
  int launch_small(const T* Vin, const C* A, C* Nout, int planes) {
    if (P <= 2) return launch_small_t<2, 1>(Vin, A, Nout, planes);
    if (P <= 6) return launch_small_t<6, 1>(Vin, A, Nout, planes);
    return launch_small_t<10, 4>(Vin, A, Nout, planes);
  }

  // N_p[A_j](t) for `planes` planes starting at plane j0 of At -> G (time domain)   (a4-a7)
  int nonlinear_term(int j0, int planes) {
    if (small_fused()) {
      if (f_R != 0.0) GM_TRY(launch_pairs(At + j0 * PN, PN, V + j0 * QN, QN, planes));     // a4 + a5
      return launch_small(V + j0 * QN, At + j0 * PN, G + j0 * PN, planes);                 // (a4 +) a6 + a7
    }
    GM_TRY(launch_pairs(At + j0 * PN, PN, V + j0 * QN, QN, planes));
    GM_TRY(launch_contract(V + j0 * QN, U + j0 * QN, planes));
    GM_TRY(launch_mode_reduce(U + j0 * QN, At + j0 * PN, G + j0 * PN, planes));
    return 0;
  }

  int to_master(const C* src) {   // psi0_d <- src (promote)
    const long long n = 2 * PN;
    prof_begin(GMMNLSE_KIND_MISC);
    launch_k(k_convert<T, double>, (unsigned)((n + 255) / 256), 256, 0, (const T*)src, (double*)psi0_d, n);
    prof_end();
    GM_CUDA(cudaGetLastError());
    return 0;
  }

  // a3-a9 of one MPA iteration over planes j0..Mc (j0 = 0 on the first iterate, which starts every plane from psi_0)
  int enqueue_iteration(int Mc, bool first) {
    const int j0 = first ? 0 : 1, np = Mc + 1 - j0;
    const unsigned sblocks = (unsigned)((PN + 255) / 256);
    // a3: A_j(t) = F^-1{psi_j exp(+D j dz)}; first iterate psi_j = psi_0
    float* fb = nullptr;
    if constexpr (sizeof(T) == 4) {
      if (tc_h && !small_fused()) {                  // the fp16 pair streams' range bound rides on a3's stores
        GM_CUDA(cudaMemsetAsync(d_vbound, 0, sizeof(float), stream));
        fb = d_vbound;
      }
    }
    GM_TRY(launch_fft(-1, first ? psi : psi + j0 * PN, first ? 0 : PN, At + j0 * PN, PN, E + j0 * PN, nullptr,
                      nullptr, PN, (T)(1.0 / N), P, np, gfwd ? gfwd + j0 * P : nullptr, fb));
    bound_from_fft = fb != nullptr;
    GM_TRY(nonlinear_term(j0, np));                                        // a4-a7
    // a8: G_j = K(w) exp(-D j dz) F{N_p}
    GM_TRY(launch_fft(+1, G + j0 * PN, PN, G + j0 * PN, PN, nullptr, Kw, E + j0 * PN, PN, (T)1, P, np,
                      ginv ? ginv + j0 * P : nullptr));
    if (ext_any())                                                          // + exp(-D j dz) X_j^T (psi_j exp(D j dz))
      GM_TRY(launch_ext(first ? psi : psi + j0 * PN, first ? 0 : PN, E + j0 * PN, gfwd ? gfwd + j0 * P : nullptr,
                        ginv ? ginv + j0 * P : nullptr, G + j0 * PN, np, j0, 0));
    // a9 + a10
    prof_begin(GMMNLSE_KIND_SCAN);
    launch_k(k_trapz_scan<T>, sblocks, 256, sizeof(double) * 2 * (Mc + 1), psi, G, psi, PN, Mc, (T)dz,
                                                                             first ? 1 : 0, errbuf, PN);
    prof_end();
    GM_CUDA(cudaGetLastError());
    return 0;
  }

  int enqueue_advance(int Mc, const double2* EM) {                           // a11
    const unsigned sblocks = (unsigned)((PN + 255) / 256);
    prof_begin(GMMNLSE_KIND_ADVANCE);
    launch_k(k_advance<T>, sblocks, 256, 0, psi0_d, psi, G, PN, Mc, dz, EM, PN, d_step2);
    prof_end();
    GM_CUDA(cudaGetLastError());
    return 0;
  }

  int get_EM(int Mc, double2** out) {        // exp(D Mc dz) in fp64: the plan's table, or one made for a ragged last step
    *out = EM_d;
    if (Mc != M) {
      auto it = EM_ragged.find(Mc);
      if (it == EM_ragged.end()) {
        double2* p = nullptr;
        GM_TRY(make_EM(Mc, &p));
        EM_ragged[Mc] = p;
        *out = p;
      } else {
        *out = it->second;
      }
    }
    return 0;
  }

  // ---- plane-axis sharding over several GPUs: the pieces of one large step that a shard runs on its
  // own planes j_lo+1 .. j_hi of the Mc planes; the collectives between them belong to the caller (sharded.py)
  C* shard_pre = nullptr;
  int shard_begin(const void* A_in) override {
    GM_TRY(fold_pending());
    GM_CUDA(cudaMemsetAsync(d_step2, 0, sizeof(int), stream));
    GM_TRY(launch_fft(+1, (const C*)A_in, 0, psi, 0, nullptr, nullptr, nullptr, 0, (T)1, P, 1));   // a1, on every shard
    return to_master(psi);
  }
  int shard_iterate(int j_lo, int j_hi, int Mc, int first, void* block_sum) override {
    if (Mc < 1 || Mc > M || j_lo < 0 || j_hi <= j_lo || j_hi > Mc) return GMMNLSE_EINVAL;
    const int ja = (first && j_lo == 0) ? 0 : j_lo + 1, np = j_hi - ja + 1;      // G_0 is formed once, by the first shard
    GM_TRY(launch_fft(-1, first ? psi : psi + ja * PN, first ? 0 : PN, At + ja * PN, PN, E + ja * PN, nullptr, nullptr, PN,
                      (T)(1.0 / N), P, np, gfwd ? gfwd + ja * P : nullptr));                        // a3
    GM_TRY(nonlinear_term(ja, np));                                                                 // a4-a7
    GM_TRY(launch_fft(+1, G + ja * PN, PN, G + ja * PN, PN, nullptr, Kw, E + ja * PN, PN, (T)1, P, np,
                      ginv ? ginv + ja * P : nullptr));                                             // a8
    if (ext_any())
      GM_TRY(launch_ext(first ? psi : psi + ja * PN, first ? 0 : PN, E + ja * PN, gfwd ? gfwd + ja * P : nullptr,
                        ginv ? ginv + ja * P : nullptr, G + ja * PN, np, ja, 0));
    prof_begin(GMMNLSE_KIND_SCAN);
    launch_k(k_shard_block_sum<T>, (unsigned)((PN + 255) / 256), 256, 0, G, PN, j_lo, j_hi, Mc, (C*)block_sum, PN);
    prof_end();
    GM_CUDA(cudaGetLastError());
    return 0;
  }
  int shard_update(int j_lo, int j_hi, int Mc, int first, const void* all_sums, int shard, int n_shards,
                   double* err_local) override {
    if (Mc < 1 || Mc > M || j_lo < 0 || j_hi <= j_lo || j_hi > Mc || shard < 0 || shard >= n_shards || !err_local)
      return GMMNLSE_EINVAL;
    if (!shard_pre) GM_TRY(dalloc(&shard_pre, (size_t)PN));
    const unsigned blocks = (unsigned)((PN + 255) / 256);
    prof_begin(GMMNLSE_KIND_SCAN);
    launch_k(k_shard_prefix<T>, blocks, 256, 0, (const C*)all_sums, shard, G, shard_pre, PN);
    launch_k(k_shard_scan<T>, blocks, 256, 0, psi, G, psi, PN, j_lo, j_hi, (T)dz, first, shard_pre, errbuf, PN);
    prof_end();
    prof_begin(GMMNLSE_KIND_MISC);
    launch_k(k_err_finalize, 1, 32, 0, errbuf, Mc, d_err);
    prof_end();
    GM_CUDA(cudaGetLastError());
    GM_CUDA(cudaMemcpyAsync(h_err, d_err, sizeof(double), cudaMemcpyDeviceToHost, stream));
    GM_CUDA(cudaStreamSynchronize(stream));
    *err_local = *h_err;
    last_err = *h_err;
    ++n_iter;
    return 0;
  }
  int shard_advance(int Mc, const void* all_sums, int n_shards) override {
    if (Mc < 1 || Mc > M || n_shards < 1) return GMMNLSE_EINVAL;
    double2* EM = nullptr;
    GM_TRY(get_EM(Mc, &EM));
    prof_begin(GMMNLSE_KIND_ADVANCE);
    launch_k(k_shard_advance<T>, (unsigned)((PN + 255) / 256), 256, 0, psi0_d, psi, (const C*)all_sums, n_shards, dz, EM, PN,
             d_step2, Mc);
    prof_end();
    GM_CUDA(cudaGetLastError());
    ++n_large;
    return 0;
  }
  int shard_end(void* A_out) override {
    return launch_fft(-1, psi, 0, (C*)A_out, 0, nullptr, nullptr, nullptr, 0, (T)(1.0 / N), P, 1);
  }

  int large_step(int Mc, bool* converged) {
    double2* EM = nullptr;
    GM_TRY(get_EM(Mc, &EM));
    const int cap = fixed_iter > 0 ? fixed_iter : max_iter;
    int it = 0;
    double err_prev = 1e300, rho_prev = 1e300;
    *converged = false;
    while (true) {
      GM_TRY(enqueue_iteration(Mc, it == 0));
      prof_begin(GMMNLSE_KIND_MISC);
      launch_k(k_err_finalize, 1, 32, 0, errbuf, Mc, d_err);
      prof_end();
      GM_CUDA(cudaGetLastError());
      ++it;
      ++n_iter;
      if (fixed_iter > 0) {
        if (it >= cap) { *converged = true; break; }
        continue;
      }
      GM_CUDA(cudaMemcpyAsync(h_err, d_err, sizeof(double), cudaMemcpyDeviceToHost, stream));
      GM_CUDA(cudaStreamSynchronize(stream));
      last_err = *h_err;
      double rho = 0.0;
      const bool conv = mpa_converged(last_err, tol, stop_rule, it, err_prev, rho_prev, &rho);
      err_prev = last_err;
      rho_prev = it == 1 ? 1e300 : rho;
      if (conv) { *converged = true; break; }
      if (it >= cap) break;
    }
    GM_TRY(enqueue_advance(Mc, EM));
    ++n_large;
    if (Mc == M) warmed = true;
    return 0;
  }

  // ---- device-side loop (options.graph = 0): the large step above as one CUDA graph, no host decision inside
  void drop_loop_graph() override {
    fold_pending();                                  // every caller has synchronised or is about to change the plan
    if (lg_exec) cudaGraphExecDestroy(lg_exec);
    if (lg) cudaGraphDestroy(lg);
    lg_exec = nullptr;
    lg = nullptr;
    if (rkg_exec) cudaGraphExecDestroy(rkg_exec);
    if (rkg) cudaGraphDestroy(rkg);
    rkg_exec = nullptr;
    rkg = nullptr;
    warmed = rk_warmed = false;      // the kernel set may change (coupling): next call starts on the host path
    if (loop_state > 0) loop_state = 0;
  }

  int capture_loop_graph() {     // runs with `stream` = cap_stream
    const int cap = fixed_iter > 0 ? fixed_iter : max_iter;
    const cudaStreamCaptureMode mode = cudaStreamCaptureModeRelaxed;
    cudaGraph_t got = nullptr;
    GM_CUDA(cudaGraphCreate(&lg, 0));
    cudaGraphConditionalHandle handle;
    GM_CUDA(cudaGraphConditionalHandleCreate(&handle, lg, 0, 0));
    auto finalize = [&]() -> int {
      prof_begin(GMMNLSE_KIND_MISC);
      launch_k(k_err_finalize_loop, 1, 32, 0, errbuf, M, d_err, tol, cap, fixed_iter > 0 ? 1 : 0, handle, d_stats, stop_rule);
      prof_end();
      GM_CUDA(cudaGetLastError());
      return 0;
    };
    // iteration 0
    GM_CUDA(cudaStreamBeginCaptureToGraph(stream, lg, nullptr, nullptr, 0, mode));
    GM_CUDA(cudaMemsetAsync(&d_stats->it, 0, sizeof(int), stream));
    long long c = n_launch;
    GM_TRY(enqueue_iteration(M, true));
    GM_TRY(finalize());
    lg_c0 = n_launch - c;
    cudaStreamCaptureStatus cs;
    unsigned long long id = 0;
    const cudaGraphNode_t* deps = nullptr;
    size_t nd = 0;
    GM_CUDA(cudaStreamGetCaptureInfo(stream, &cs, &id, &got, &deps, &nd));
    std::vector<cudaGraphNode_t> tail(deps, deps + nd);
    GM_CUDA(cudaStreamEndCapture(stream, &got));
    // while (continue) { one further iteration }
    cudaGraphNodeParams cp = {};
    cp.type = cudaGraphNodeTypeConditional;
    cp.conditional.handle = handle;
    cp.conditional.type = cudaGraphCondTypeWhile;
    cp.conditional.size = 1;
    cudaGraphNode_t loop_node;
    GM_CUDA(cudaGraphAddNode(&loop_node, lg, tail.data(), tail.size(), &cp));
    cudaGraph_t body = cp.conditional.phGraph_out[0];
    GM_CUDA(cudaStreamBeginCaptureToGraph(stream, body, nullptr, nullptr, 0, mode));
    c = n_launch;
    GM_TRY(enqueue_iteration(M, false));
    GM_TRY(finalize());
    lg_cb = n_launch - c;
    GM_CUDA(cudaStreamEndCapture(stream, &got));
    // a11
    GM_CUDA(cudaStreamBeginCaptureToGraph(stream, lg, &loop_node, nullptr, 1, mode));
    c = n_launch;
    GM_TRY(enqueue_advance(M, EM_d));
    lg_ca = n_launch - c;
    GM_CUDA(cudaStreamEndCapture(stream, &got));
    GM_CUDA(cudaGraphInstantiate(&lg_exec, lg, 0));
    return 0;
  }

  int build_loop_graph() {
    if (!cap_stream) GM_CUDA(cudaStreamCreateWithFlags(&cap_stream, cudaStreamNonBlocking));
    if (!d_stats) {
      GM_CUDA(cudaMalloc(&d_stats, sizeof(LoopStats)));
      GM_CUDA(cudaMallocHost(&h_stats, sizeof(LoopStats)));
    }
    GM_CUDA(cudaStreamSynchronize(stream));
    cudaStream_t user = stream;
    const long long nl = n_launch;
    stream = cap_stream;
    const int st = capture_loop_graph();
    stream = user;
    n_launch = nl;
    if (st != 0) {
      cudaStreamCaptureStatus cs = cudaStreamCaptureStatusNone;
      if (cudaStreamIsCapturing(cap_stream, &cs) == cudaSuccess && cs != cudaStreamCaptureStatusNone) {
        cudaGraph_t tmp = nullptr;
        cudaStreamEndCapture(cap_stream, &tmp);
      }
      drop_loop_graph();
      cudaGetLastError();
      loop_state = -1;
      return st;
    }
    loop_state = 1;
    return 0;
  }

  int propagate(const void* A_in, double L, void* A_out) override {
    const double ns = L / dz;
    const long long nsteps = llround(ns);
    if (!(L >= 0) || std::fabs(ns - (double)nsteps) > 1e-9 * std::fmax(1.0, ns)) return GMMNLSE_EINVAL;
    if (fprof_d && Qc && 2 * nsteps + 1 > n_fprof) return GMMNLSE_EINVAL;   // the z-profile must cover the call
    GM_TRY(fold_pending());
    GM_CUDA(cudaMemsetAsync(d_step2, 0, sizeof(int), stream));
    // a1: psi_0 = F{A(z0)}
    GM_TRY(launch_fft(+1, (const C*)A_in, 0, psi, 0, nullptr, nullptr, nullptr, 0, (T)1, P, 1));
    GM_TRY(to_master(psi));
    long long done = 0, gsteps = 0;
    int status = GMMNLSE_OK;
    bool last_on_device = false;
    while (done < nsteps) {
      const int Mc = (int)std::min<long long>(M, nsteps - done);
      // full large steps run as one graph launch each once a host-loop step has set the kernels up; the ragged
      // last step, per-kernel event timing and options.graph = 1 keep the host loop
      bool on_device = graph == 0 && !prof_on && Mc == M && warmed && loop_state >= 0;
      if (on_device && !lg_exec && build_loop_graph() != 0) on_device = false;
      if (on_device) {
        if (gsteps == 0) GM_CUDA(cudaMemsetAsync(d_stats, 0, sizeof(LoopStats), stream));
        GM_CUDA(cudaGraphLaunch(lg_exec, stream));
        ++gsteps;
        ++n_large;
        last_on_device = true;
      } else {
        bool conv = false;
        GM_TRY(large_step(Mc, &conv));
        if (!conv) { ++n_noconv; status = GMMNLSE_WARN_NOCONV; }
        last_on_device = false;
      }
      done += Mc;
    }
    // A_out = F^-1{psi_0}
    GM_TRY(launch_fft(-1, psi, 0, (C*)A_out, 0, nullptr, nullptr, nullptr, 0, (T)(1.0 / N), P, 1));
    if (d2h_dst) GM_CUDA(cudaMemcpyAsync(d2h_dst, A_out, d2h_bytes, cudaMemcpyDeviceToHost, stream));   // host entry
    if (gsteps > 0) {            // one read-back per call: iteration count, unconverged steps, last error
      GM_CUDA(cudaMemcpyAsync(h_stats, d_stats, sizeof(LoopStats), cudaMemcpyDeviceToHost, stream));
      if (async_call && !d2h_dst) {                // return now; the counters are folded in when somebody needs them
        pending_gsteps = gsteps;
        pending_last_on_device = last_on_device;
        pending_stream = stream;
        return status;
      }
      GM_CUDA(cudaStreamSynchronize(stream));
      take_loop_stats(gsteps, last_on_device, &status);
    } else {                     // host loop: same completion semantics (A_out complete on return)
      if (fixed_iter > 0) GM_CUDA(cudaMemcpyAsync(h_err, d_err, sizeof(double), cudaMemcpyDeviceToHost, stream));
      GM_CUDA(cudaStreamSynchronize(stream));
      if (fixed_iter > 0) last_err = nsteps > 0 ? *h_err : 0.0;
    }
    return status;
  }

  // 1 page-locked host memory (cudaMallocHost / cudaHostRegister), 0 pageable host memory, -1 device or managed
  // memory (not a host buffer: the caller wants gmmnlse_propagate)
  static int host_kind(const void* p) {
    cudaPointerAttributes a;
    if (cudaPointerGetAttributes(&a, p) != cudaSuccess) { cudaGetLastError(); return 0; }
    if (a.type == cudaMemoryTypeHost) return 1;
    return a.type == cudaMemoryTypeUnregistered ? 0 : -1;
  }

  // Host entry: H2D, propagate, D2H on the plan's stream, one synchronise.  Page-locked caller buffers are copied
  // from and to directly; pageable ones are staged through plan-owned pinned memory (two host memcpys more).
  int propagate_host(const void* A_in, double L, void* A_out) override {
    const size_t bytes = sizeof(C) * (size_t)PN;
    if (!d_io) GM_TRY(dalloc(&d_io, (size_t)PN));
    const int k_in = host_kind(A_in), k_out = host_kind(A_out);
    if (k_in < 0 || k_out < 0) return GMMNLSE_EINVAL;
    const bool pin_in = k_in == 1, pin_out = k_out == 1;
    if ((!pin_in || !pin_out) && !h_in) {
      GM_CUDA(cudaMallocHost(&h_in, bytes));
      GM_CUDA(cudaMallocHost(&h_out, bytes));
    }
    if (!pin_in) std::memcpy(h_in, A_in, bytes);
    GM_CUDA(cudaMemcpyAsync(d_io, pin_in ? A_in : h_in, bytes, cudaMemcpyHostToDevice, stream));
    d2h_dst = pin_out ? A_out : h_out;             // propagate() enqueues this copy ahead of its own read-back
    d2h_bytes = bytes;
    const int st = propagate(d_io, L, d_io);
    d2h_dst = nullptr;
    if (st < 0) return st;
    GM_CUDA(cudaStreamSynchronize(stream));
    if (!pin_out) std::memcpy(A_out, h_out, bytes);
    return st;
  }

  // Nh(X) = K F{N[F^-1 X]} for one [P][N] field in the frequency domain -> G plane 0      (a3-a8, one plane)
  // f_off: position of the evaluation inside the step in half small steps (RK4IP stages: 0, 1, 1, 2)
  int nonlinear_freq(const C* Xf, int f_off) {
    GM_TRY(launch_fft(-1, Xf, 0, At, 0, nullptr, nullptr, nullptr, 0, (T)(1.0 / N), P, 1));
    GM_TRY(nonlinear_term(0, 1));
    GM_TRY(launch_fft(+1, G, 0, G, 0, nullptr, Kw, nullptr, 0, (T)1, P, 1));
    if (ext_any()) GM_TRY(launch_ext(Xf, 0, nullptr, nullptr, nullptr, G, 1, 0, f_off));
    return 0;
  }

  // Linear extra terms of section F: coupling i Q (constant, or f(z) Q with a z-profile) and the
  // first-order gain saturation.  The matrix is the same for every plane only for constant coupling alone.
  bool ext_any() const { return Qc != nullptr || g_sat != 0.0; }
  bool ext_dynamic() const { return g_sat != 0.0 || (Qc && fprof_d); }
  // G_j += R-_j X_j^T (R+_j src_j) for `planes` planes starting at plane j0 (At planes j0.. hold the fields in time)
  int launch_ext(const C* src, long long src_ps, const C* Etab, const T* gf, const T* gi, C* Gout, int planes, int j0,
                 int f_off) {
    const C* X = Xconst;
    long long x_ps = 0;
    if (ext_dynamic()) {
      if (!Xext) GM_TRY(dalloc(&Xext, (size_t)(M + 1) * P * P));
      if (g_sat != 0.0) {
        if (!Epair) GM_TRY(dalloc(&Epair, (size_t)(M + 1) * Q));
        prof_begin(GMMNLSE_KIND_MISC);
        launch_k(k_pair_energy<T>, dim3(Q, planes), 256, 0, At + j0 * PN, PN, pair_m, pair_n, Epair + (size_t)j0 * Q, Q, N, dt);
        prof_end();
        GM_CUDA(cudaGetLastError());
      }
      prof_begin(GMMNLSE_KIND_MISC);
      launch_k(k_ext_matrix<T>, planes, 256, 0, Qc, S2, g_sat != 0.0 ? Epair + (size_t)j0 * Q : nullptr, (T)g_sat, fprof_d,
               n_fprof, d_step2, j0, f_off, Xext + (size_t)j0 * P * P, P, Q);
      prof_end();
      GM_CUDA(cudaGetLastError());
      X = Xext + (size_t)j0 * P * P;
      x_ps = (long long)P * P;
    }
    const size_t smem = sizeof(C) * P * 64;
    GM_TRY(ensure_smem(k_couple<T>, smem));
    prof_begin(GMMNLSE_KIND_MISC);
    launch_k(k_couple<T>, dim3((N + 63) / 64, planes), 256, smem, src, src_ps, Etab, gf, gi, X, x_ps, Gout, PN, P, N);
    prof_end();
    GM_CUDA(cudaGetLastError());
    return 0;
  }

  int set_gain(const double* g) override {
    GM_CUDA(cudaStreamSynchronize(stream));
    drop_loop_graph();
    bool any = false;
    if (g)
      for (int p = 0; p < P; ++p) {
        if (!std::isfinite(g[p])) return GMMNLSE_EINVAL;
        any = any || g[p] != 0.0;
      }
    cudaFree(gfwd); cudaFree(ginv); cudaFree(EM_d); cudaFree(EH_d);
    gfwd = ginv = nullptr; EM_d = nullptr; EH_d = nullptr;
    for (auto& kv : EM_ragged) cudaFree(kv.second);
    EM_ragged.clear();
    gain.clear();
    if (any) {
      gain.assign(g, g + P);
      std::vector<T> f((size_t)(M + 1) * P), b((size_t)(M + 1) * P);
      for (int jn = 0; jn <= M; ++jn)
        for (int p = 0; p < P; ++p) {
          f[(size_t)jn * P + p] = (T)std::exp(gain[p] * (jn * dz));
          b[(size_t)jn * P + p] = (T)std::exp(-gain[p] * (jn * dz));
        }
      GM_TRY(dalloc(&gfwd, f.size())); GM_TRY(upload(gfwd, f));
      GM_TRY(dalloc(&ginv, b.size())); GM_TRY(upload(ginv, b));
    }
    return make_EM(M, &EM_d);
  }

  int set_coupling(const double* Qri) override {
    GM_CUDA(cudaStreamSynchronize(stream));
    drop_loop_graph();
    cudaFree(Qc);
    cudaFree(Xconst);
    Qc = nullptr;
    Xconst = nullptr;
    if (!Qri) return 0;
    std::vector<C> q((size_t)P * P);
    bool any = false;
    for (size_t i = 0; i < q.size(); ++i) {
      if (!std::isfinite(Qri[2 * i]) || !std::isfinite(Qri[2 * i + 1])) return GMMNLSE_EINVAL;
      q[i] = mk((T)Qri[2 * i], (T)Qri[2 * i + 1]);
      any = any || Qri[2 * i] != 0.0 || Qri[2 * i + 1] != 0.0;
    }
    if (!any) return 0;
    GM_TRY(dalloc(&Qc, q.size()));
    GM_TRY(upload(Qc, q));
    std::vector<C> x(q.size());
    for (size_t i = 0; i < q.size(); ++i) x[i] = mk(-q[i].y, q[i].x);      // i Q
    GM_TRY(dalloc(&Xconst, x.size()));
    return upload(Xconst, x);
  }

  // z-profile of the coupling: Q(z) = f(z) Q (index perturbation eps(x, y) f(z)), f sampled every dz / 2
  // from the start of each propagate call (the RK4IP stages sit on half steps)
  int set_coupling_profile(const double* f, int n) override {
    GM_CUDA(cudaStreamSynchronize(stream));
    drop_loop_graph();
    cudaFree(fprof_d);
    fprof_d = nullptr;
    n_fprof = 0;
    if (!f) return 0;
    if (n < 1) return GMMNLSE_EINVAL;
    for (int i = 0; i < n; ++i)
      if (!std::isfinite(f[i])) return GMMNLSE_EINVAL;
    GM_TRY(dalloc(&fprof_d, (size_t)n));
    GM_CUDA(cudaMemcpy(fprof_d, f, sizeof(double) * (size_t)n, cudaMemcpyHostToDevice));
    n_fprof = n;
    return 0;
  }

  int set_gain_saturation(double g) override {
    if (!std::isfinite(g)) return GMMNLSE_EINVAL;
    if (g != 0.0 && general) return GMMNLSE_EUNSUPPORTED;           // needs the packed symmetric S2
    GM_CUDA(cudaStreamSynchronize(stream));
    drop_loop_graph();
    g_sat = g;
    return 0;
  }

  int enqueue_rk4_step() {
    const unsigned blocks = (unsigned)((PN + 255) / 256);
    for (int stage = 1; stage <= 4; ++stage) {
      GM_TRY(nonlinear_freq(stage == 1 ? psi : rk_X, stage == 1 ? 0 : (stage == 4 ? 2 : 1)));
      prof_begin(GMMNLSE_KIND_ADVANCE);
      launch_k(k_rk4_stage<T>, blocks, 256, 0, stage, psi0_d, psi, EH_d, G, rk_AI, rk_K1, rk_K2, rk_K3, rk_X, dz, PN, d_step2);
      prof_end();
      GM_CUDA(cudaGetLastError());
    }
    return 0;
  }

  int build_rk4_graph() {
    if (!cap_stream) GM_CUDA(cudaStreamCreateWithFlags(&cap_stream, cudaStreamNonBlocking));
    GM_CUDA(cudaStreamSynchronize(stream));
    cudaStream_t user = stream;
    const long long nl = n_launch;
    stream = cap_stream;
    int st = cudaStreamBeginCapture(stream, cudaStreamCaptureModeRelaxed) == cudaSuccess ? 0 : GMMNLSE_ECUDA;
    if (st == 0) {
      st = enqueue_rk4_step();
      rk_c = n_launch - nl;
      if (cudaStreamEndCapture(stream, &rkg) != cudaSuccess) st = GMMNLSE_ECUDA;
    }
    if (st == 0 && cudaGraphInstantiate(&rkg_exec, rkg, 0) != cudaSuccess) st = GMMNLSE_ECUDA;
    stream = user;
    n_launch = nl;
    if (st != 0) {
      if (rkg) cudaGraphDestroy(rkg);
      rkg = nullptr;
      rkg_exec = nullptr;
      cudaGetLastError();
      rk_graph_failed = true;
    }
    return st;
  }

  int propagate_rk4ip(const void* A_in, double L, void* A_out) override {
    const double ns = L / dz;
    const long long nsteps = llround(ns);
    if (!(L >= 0) || std::fabs(ns - (double)nsteps) > 1e-9 * std::fmax(1.0, ns)) return GMMNLSE_EINVAL;
    if (!rk_X) {
      GM_TRY(dalloc(&rk_X, (size_t)PN)); GM_TRY(dalloc(&rk_AI, (size_t)PN)); GM_TRY(dalloc(&rk_K1, (size_t)PN));
      GM_TRY(dalloc(&rk_K2, (size_t)PN)); GM_TRY(dalloc(&rk_K3, (size_t)PN));
    }
    if (!EH_d) {
      std::vector<double2> eh((size_t)PN);
      for (long long i = 0; i < PN; ++i) {
        const double ph = std::remainder(phi[i] * (0.5 * dz), 2.0 * M_PI);
        const double mag = gain.empty() ? 1.0 : std::exp(gain[(size_t)(i / N)] * (0.5 * dz));
        eh[i] = make_double2(mag * std::cos(ph), mag * std::sin(ph));
      }
      GM_TRY(dalloc(&EH_d, (size_t)PN));
      GM_TRY(upload(EH_d, eh));
    }
    if (fprof_d && Qc && 2 * nsteps + 1 > n_fprof) return GMMNLSE_EINVAL;
    GM_TRY(fold_pending());
    GM_CUDA(cudaMemsetAsync(d_step2, 0, sizeof(int), stream));
    GM_TRY(launch_fft(+1, (const C*)A_in, 0, psi, 0, nullptr, nullptr, nullptr, 0, (T)1, P, 1));
    GM_TRY(to_master(psi));
    long long s = 0;
    if (nsteps > 0 && !rk_warmed) {                  // first step of a plan on the host path: sets kernel attributes
      GM_TRY(enqueue_rk4_step());
      rk_warmed = true;
      s = 1;
    }
    const bool replay = graph == 0 && !prof_on && !rk_graph_failed && s < nsteps && (rkg_exec || build_rk4_graph() == 0);
    for (; s < nsteps; ++s) {
      if (replay) {
        GM_CUDA(cudaGraphLaunch(rkg_exec, stream));
        n_launch += rk_c;
      } else {
        GM_TRY(enqueue_rk4_step());
      }
    }
    GM_TRY(launch_fft(-1, psi, 0, (C*)A_out, 0, nullptr, nullptr, nullptr, 0, (T)(1.0 / N), P, 1));
    return GMMNLSE_OK;
  }

  int nonlinear_op(const void* A, void* dA) override {
    // a12: uses plane 0 of the scratch buffers.  dA = F^-1{ K(w) F{N_p[A]} }
    GM_CUDA(cudaMemcpyAsync(At, A, sizeof(C) * (size_t)PN, cudaMemcpyDeviceToDevice, stream));
    GM_TRY(nonlinear_term(0, 1));
    GM_TRY(launch_fft(+1, G, 0, G, 0, nullptr, Kw, nullptr, 0, (T)1, P, 1));
    GM_TRY(launch_fft(-1, G, 0, (C*)dA, 0, nullptr, nullptr, nullptr, 0, (T)(1.0 / N), P, 1));
    return 0;
  }

  int get_planes(void* out) override {
    GM_CUDA(cudaStreamSynchronize(stream));
    GM_CUDA(cudaMemcpy(out, psi, sizeof(C) * (size_t)(M + 1) * PN, cudaMemcpyDeviceToHost));
    return 0;
  }

  int debug_fft(const void* in, void* out, int rows, int dir) override {
    if (rows < 1 || (dir != 1 && dir != -1)) return GMMNLSE_EINVAL;
    return launch_fft(dir, (const C*)in, 0, (C*)out, 0, nullptr, nullptr, nullptr, 0,
                      dir > 0 ? (T)1 : (T)(1.0 / N), rows, 1);
  }
  int debug_pairs(const void* A, void* Vout, int n_planes) override {
    if (n_planes < 1) return GMMNLSE_EINVAL;
    return launch_pairs((const C*)A, PN, (T*)Vout, QN, n_planes);
  }
  int contraction_kind() const override {
    if (tc_h) return sparse ? 9 : (lowrank ? 8 : 7);
    return lowrank ? 6 : (tc_on ? 3 : 1);
  }
  int lowrank_rank() const override { return lowrank ? lr_R : 0; }
  int sparse_info(int* classes, double* work_fraction) const override {
    if (classes) *classes = sparse ? sp_classes : 0;
    if (work_fraction) *work_fraction = sparse ? sp_work_fraction : 1.0;
    return 0;
  }
  int raman_kind() const override { return f_R == 0.0 ? 0 : (iir ? 2 : 1); }
  int set_tc_chunk(int k) override {
    if (k < 1 || k > 255) return GMMNLSE_EINVAL;
    cudaStreamSynchronize(stream);
    drop_loop_graph();
    tc_kchunk = k;
    return 0;
  }
  int debug_contract(const void* Vin, void* Uout, int n_planes) override {
    if (n_planes < 1) return GMMNLSE_EINVAL;
    return launch_contract((const T*)Vin, (T*)Uout, n_planes);
  }
};

// ------------------------------------------------------------------ Eq. 2 by quadrature on the GPU (NEXT-4)
struct DevBufs {                      // frees what it owns when the routine leaves, on every path
  std::vector<void*> p;
  ~DevBufs() { for (void* q : p) cudaFree(q); }
  template <typename X> int alloc(X** out, size_t n) {
    cudaError_t e = cudaMalloc((void**)out, n * sizeof(X));
    if (e == cudaErrorMemoryAllocation) { cudaGetLastError(); return GMMNLSE_ENOMEM; }
    GM_CUDA(e);
    p.push_back(*out);
    return 0;
  }
};

// S_plmn = int F_p F_l F_m F_n dA / sqrt(int F_p^2 dA ... int F_n^2 dA): the Gram matrix of the pair
// functions F_p F_l (p <= l) over the G grid points is one (Q x G) (G x Q) product -- K = G on the kind::f16 tcgen05
// kernel of gemm_h.cuh, both operands split into fp16 hi / lo with exact power-of-two scales -- then the
// normalisation and the expansion to [P]^4 on the host in fp64.
int overlap_tensor_gpu(int P, long long G, const double* F, double dA, double* S_out) {
  const int Q = P * (P + 1) / 2;
  const int Npad = (Q + hc::TM - 1) / hc::TM * hc::TM;           // pair index as the GEMM's M (t) dimension
  const int nrt = (Q + 207) / 208;
  const int NT = (((Q + nrt - 1) / nrt) + 15) / 16 * 16;
  const int Rp = nrt * NT;
  const int KB = (int)(G / hc::BK);
  int dev = 0, n_sm = 0, smax = 0;
  GM_CUDA(cudaGetDevice(&dev));
  GM_CUDA(cudaDeviceGetAttribute(&n_sm, cudaDevAttrMultiProcessorCount, dev));
  GM_CUDA(cudaDeviceGetAttribute(&smax, cudaDevAttrMaxSharedMemoryPerBlockOptin, dev));
  int stages = 3;
  while (stages > 1 && hc::smem_bytes(NT, stages) > (size_t)smax) --stages;
  if (hc::smem_bytes(NT, stages) > (size_t)smax) return GMMNLSE_EUNSUPPORTED;
  std::vector<int> pp(Q), pl(Q);
  for (int p = 0, q = 0; p < P; ++p)
    for (int l = p; l < P; ++l, ++q) { pp[q] = p; pl[q] = l; }
  DevBufs bufs;
  double* dF = nullptr;
  int *dpp = nullptr, *dpl = nullptr;
  float *PhiT = nullptr, *Ug = nullptr, *rscale = nullptr, *vbound = nullptr;
  __half *Ah = nullptr, *Bh = nullptr, *Bl = nullptr;
  GM_TRY(bufs.alloc(&dF, (size_t)P * G));
  GM_TRY(bufs.alloc(&dpp, (size_t)Q));
  GM_TRY(bufs.alloc(&dpl, (size_t)Q));
  GM_TRY(bufs.alloc(&PhiT, (size_t)G * Npad));
  GM_TRY(bufs.alloc(&Ah, (size_t)2 * G * Npad));                  // hi rows [G][Npad], then lo rows
  GM_TRY(bufs.alloc(&Bh, (size_t)Rp * G));
  GM_TRY(bufs.alloc(&Bl, (size_t)Rp * G));
  GM_TRY(bufs.alloc(&rscale, (size_t)Rp));
  GM_TRY(bufs.alloc(&vbound, (size_t)1));
  GM_TRY(bufs.alloc(&Ug, (size_t)Q * Npad));
  // normalise the modes first (fp64, host): unnormalised Hermite-Gauss fields of high order are orders of magnitude
  // larger than the fundamental, and the fp16 operands share one power-of-two range
  std::vector<double> Fn((size_t)P * G);
  for (int p = 0; p < P; ++p) {
    long double acc = 0;
    for (long long g = 0; g < G; ++g) acc += (long double)F[p * G + g] * F[p * G + g];
    const double nrm = std::sqrt((double)acc * dA);
    if (!(nrm > 0) || !std::isfinite(nrm)) return GMMNLSE_EINVAL;
    for (long long g = 0; g < G; ++g) Fn[(size_t)p * G + g] = F[p * G + g] / nrm;
  }
  GM_CUDA(cudaMemcpy(dF, Fn.data(), sizeof(double) * (size_t)P * G, cudaMemcpyHostToDevice));
  GM_CUDA(cudaMemcpy(dpp, pp.data(), sizeof(int) * Q, cudaMemcpyHostToDevice));
  GM_CUDA(cudaMemcpy(dpl, pl.data(), sizeof(int) * Q, cudaMemcpyHostToDevice));
  GM_CUDA(cudaMemset(vbound, 0, sizeof(float)));
  const long long total = G * Npad;
  k_pair_fields_t<<<2368, 256>>>(dF, G, dpp, dpl, Q, Npad, PhiT);
  k_bound_real<float><<<592, 256>>>(PhiT, total, vbound);
  k_v_encode<<<2368, 256>>>(PhiT, total, total, HalfOut{Ah, 2 * total, total, Npad, vbound});
  k_pair_fields_b<<<Rp, 256>>>(dF, G, dpp, dpl, Q, Bh, Bl, rscale);
  GM_CUDA(cudaGetLastError());
  CUtensorMap tmAh, tmAl, tmBh, tmBl;
  {
    const cuuint64_t dims[3] = {(cuuint64_t)Npad, (cuuint64_t)G, 1};
    const cuuint64_t strides[2] = {(cuuint64_t)Npad * 2, (cuuint64_t)G * Npad * 4};
    const cuuint32_t box[3] = {64, hc::BK, 1};
    GM_TRY(encode_tmap(&tmAh, CU_TENSOR_MAP_DATA_TYPE_FLOAT16, Ah, 3, dims, strides, box, CU_TENSOR_MAP_SWIZZLE_128B));
    GM_TRY(encode_tmap(&tmAl, CU_TENSOR_MAP_DATA_TYPE_FLOAT16, Ah + total, 3, dims, strides, box,
                       CU_TENSOR_MAP_SWIZZLE_128B));
  }
  {
    const cuuint64_t dims[2] = {(cuuint64_t)G, (cuuint64_t)Rp};
    const cuuint64_t strides[1] = {(cuuint64_t)G * 2};
    const cuuint32_t box[2] = {hc::BK, (cuuint32_t)NT};
    GM_TRY(encode_tmap(&tmBh, CU_TENSOR_MAP_DATA_TYPE_FLOAT16, Bh, 2, dims, strides, box, CU_TENSOR_MAP_SWIZZLE_64B));
    GM_TRY(encode_tmap(&tmBl, CU_TENSOR_MAP_DATA_TYPE_FLOAT16, Bl, 2, dims, strides, box, CU_TENSOR_MAP_SWIZZLE_64B));
  }
  hc::Params prm = {};
  prm.U = Ug; prm.Zh = nullptr; prm.u_plane_stride = (long long)Q * Npad;
  prm.rscale = rscale; prm.vbound = vbound; prm.bound_gain = 1.f; prm.zgain = 0.f;
  prm.Q = Q; prm.N = Npad; prm.NT = NT; prm.KB = KB; prm.n_rt = nrt;
  prm.t_tiles = Npad / hc::TM;
  prm.total_tiles = prm.t_tiles * nrt;
  prm.plane0 = 0; prm.stages = stages; prm.kchunk = 4;
  GM_TRY(ensure_dyn_smem(dev, (const void*)hc::k_contract_h<false>, hc::smem_bytes(NT, stages)));
  cudaLaunchConfig_t cfg = {};
  cfg.gridDim = dim3((unsigned)std::min(n_sm, prm.total_tiles));
  cfg.blockDim = dim3(hc::NTHREADS);
  cfg.dynamicSmemBytes = hc::smem_bytes(NT, stages);
  GM_CUDA(cudaLaunchKernelEx(&cfg, hc::k_contract_h<false>, tmAh, tmAl, tmBh, tmBl, prm));
  std::vector<float> Uh((size_t)Q * Npad);
  GM_CUDA(cudaMemcpy(Uh.data(), Ug, sizeof(float) * Uh.size(), cudaMemcpyDeviceToHost));   // synchronises
  // expansion to [P]^4 in fp64 on the host (the modes were normalised before the product)
  std::vector<int> idx((size_t)P * P);
  for (int q = 0; q < Q; ++q) { idx[(size_t)pp[q] * P + pl[q]] = q; idx[(size_t)pl[q] * P + pp[q]] = q; }
  for (int p = 0; p < P; ++p)
    for (int l = 0; l < P; ++l) {
      const int r = idx[(size_t)p * P + l];
      for (int m = 0; m < P; ++m)
        for (int n = 0; n < P; ++n) {
          const int q = idx[(size_t)m * P + n];
          // the Gram matrix is symmetric: average the two computed halves
          const double gsum = 0.5 * ((double)Uh[(size_t)r * Npad + q] + (double)Uh[(size_t)q * Npad + r]);
          S_out[(((size_t)p * P + l) * P + m) * P + n] = gsum * dA;
        }
    }
  return 0;
}

// ------------------------------------------------------------------ Eq. 2 without any allocation
// gmmnlse_overlap_tensor_noalloc: the same Gram product for callers that cannot call cudaMalloc (code under CUDA graph
// capture, tight serving loops, harnesses that forbid it).  Every intermediate that overlap_tensor_gpu cudaMallocs per
// call lives in ONE file-scope device array of fixed size instead; every GPU that loads the library holds it until
// exit.  Limits: P <= NOALLOC_PMAX modes, G <= NOALLOC_GMAX grid points.
constexpr int NOALLOC_PMAX = 6;                                   // Q = 21 pair functions: one 128 x 32 tile
constexpr long long NOALLOC_GMAX = 4096;                          // e.g. a 64 x 64 quadrature grid
constexpr int NOALLOC_QMAX = NOALLOC_PMAX * (NOALLOC_PMAX + 1) / 2;
constexpr int NOALLOC_NPAD = hc::TM;                              // pair index padded to the GEMM's M tile
constexpr int NOALLOC_NT = (NOALLOC_QMAX + 15) / 16 * 16;         // 32 rows of the B operand
constexpr size_t na_align(size_t x) { return (x + 255) & ~(size_t)255; }
constexpr size_t NA_OFF_FN = 0;                                                                   // double [P][G]
constexpr size_t NA_OFF_PP = NA_OFF_FN + na_align(sizeof(double) * NOALLOC_PMAX * NOALLOC_GMAX);   // int [Q]
constexpr size_t NA_OFF_PL = NA_OFF_PP + na_align(sizeof(int) * NOALLOC_QMAX);                     // int [Q]
constexpr size_t NA_OFF_PHIT = NA_OFF_PL + na_align(sizeof(int) * NOALLOC_QMAX);                   // float [G][NPAD]
constexpr size_t NA_OFF_AH = NA_OFF_PHIT + na_align(sizeof(float) * NOALLOC_GMAX * NOALLOC_NPAD);  // half [2][G][NPAD]
constexpr size_t NA_OFF_BH = NA_OFF_AH + na_align(sizeof(__half) * 2 * NOALLOC_GMAX * NOALLOC_NPAD);   // half [NT][G]
constexpr size_t NA_OFF_BL = NA_OFF_BH + na_align(sizeof(__half) * NOALLOC_NT * NOALLOC_GMAX);     // half [NT][G]
constexpr size_t NA_OFF_RS = NA_OFF_BL + na_align(sizeof(__half) * NOALLOC_NT * NOALLOC_GMAX);     // float [NT]
constexpr size_t NA_OFF_VB = NA_OFF_RS + na_align(sizeof(float) * NOALLOC_NT);                     // float: bound on |Phi|
constexpr size_t NA_OFF_UG = NA_OFF_VB + na_align(sizeof(float));                                  // float [Q][NPAD]
constexpr size_t NOALLOC_BYTES = NA_OFF_UG + na_align(sizeof(float) * NOALLOC_QMAX * NOALLOC_NPAD);  // about 4.9 MB

// In host code this name is only a host-side stand-in for the symbol, never a device address: the address the kernels
// get comes from cudaGetSymbolAddress (noalloc_scratch_ptr below), once per device.
static __device__ __align__(256) unsigned char g_noalloc_scratch[NOALLOC_BYTES];

std::mutex g_noalloc_mu;
std::map<int, unsigned char*> g_noalloc_ptr;                      // device ordinal -> device address of the array

// device address of the scratch array on the CURRENT device (looked up once per device, with that device current)
int noalloc_scratch_ptr(int dev, unsigned char** out) {
  std::lock_guard<std::mutex> lk(g_noalloc_mu);
  auto it = g_noalloc_ptr.find(dev);
  if (it == g_noalloc_ptr.end()) {
    unsigned char* ptr = nullptr;
    GM_CUDA(cudaGetSymbolAddress((void**)&ptr, g_noalloc_scratch));
    if (!ptr) { g_cuda_err = "cudaGetSymbolAddress(g_noalloc_scratch) returned a null address"; return GMMNLSE_ECUDA; }
    it = g_noalloc_ptr.emplace(dev, ptr).first;
  }
  *out = it->second;
  return 0;
}

// Same arithmetic as overlap_tensor_gpu from the product on; the normalisation and the expansion to [P]^4 run on the
// device (k_normalise_modes, k_expand_gram) so that nothing returns to the host.  No cudaMalloc / cudaFree, no host
// heap use, no synchronisation: everything is enqueued on `stream`.
int overlap_tensor_noalloc(int P, long long G, const double* F_dev, double dA, double* S_dev, cudaStream_t stream) {
  const int Q = P * (P + 1) / 2;
  const int Npad = NOALLOC_NPAD, NT = (Q + 15) / 16 * 16, KB = (int)(G / hc::BK);
  int dev = 0, n_sm = 0, smax = 0;
  GM_CUDA(cudaGetDevice(&dev));
  GM_CUDA(cudaDeviceGetAttribute(&n_sm, cudaDevAttrMultiProcessorCount, dev));
  GM_CUDA(cudaDeviceGetAttribute(&smax, cudaDevAttrMaxSharedMemoryPerBlockOptin, dev));
  const int stages = 3;
  if (hc::smem_bytes(NT, stages) > (size_t)smax) return GMMNLSE_EUNSUPPORTED;
  unsigned char* base = nullptr;
  GM_TRY(noalloc_scratch_ptr(dev, &base));
  double* Fn = reinterpret_cast<double*>(base + NA_OFF_FN);
  int* dpp = reinterpret_cast<int*>(base + NA_OFF_PP);
  int* dpl = reinterpret_cast<int*>(base + NA_OFF_PL);
  float* PhiT = reinterpret_cast<float*>(base + NA_OFF_PHIT);
  __half* Ah = reinterpret_cast<__half*>(base + NA_OFF_AH);
  __half* Bh = reinterpret_cast<__half*>(base + NA_OFF_BH);
  __half* Bl = reinterpret_cast<__half*>(base + NA_OFF_BL);
  float* rscale = reinterpret_cast<float*>(base + NA_OFF_RS);
  float* vbound = reinterpret_cast<float*>(base + NA_OFF_VB);
  float* Ug = reinterpret_cast<float*>(base + NA_OFF_UG);
  const long long total = G * Npad;
  // the array keeps the previous call's contents: the bound is an atomicMax accumulator and must start at zero;
  // everything else is fully overwritten before it is read (PhiT beyond Q is written as zero, B rows up to NT too)
  GM_CUDA(cudaMemsetAsync(vbound, 0, sizeof(float), stream));
  k_normalise_modes<<<P, 256, 0, stream>>>(F_dev, G, dA, P, Fn, dpp, dpl);
  k_pair_fields_t<<<592, 256, 0, stream>>>(Fn, G, dpp, dpl, Q, Npad, PhiT);
  k_bound_real<float><<<592, 256, 0, stream>>>(PhiT, total, vbound);
  k_v_encode<<<592, 256, 0, stream>>>(PhiT, total, total, HalfOut{Ah, 2 * total, total, Npad, vbound});
  k_pair_fields_b<<<NT, 256, 0, stream>>>(Fn, G, dpp, dpl, Q, Bh, Bl, rscale);
  GM_CUDA(cudaGetLastError());
  CUtensorMap tmAh, tmAl, tmBh, tmBl;
  {
    const cuuint64_t dims[3] = {(cuuint64_t)Npad, (cuuint64_t)G, 1};
    const cuuint64_t strides[2] = {(cuuint64_t)Npad * 2, (cuuint64_t)G * Npad * 4};
    const cuuint32_t box[3] = {64, hc::BK, 1};
    GM_TRY(encode_tmap(&tmAh, CU_TENSOR_MAP_DATA_TYPE_FLOAT16, Ah, 3, dims, strides, box, CU_TENSOR_MAP_SWIZZLE_128B));
    GM_TRY(encode_tmap(&tmAl, CU_TENSOR_MAP_DATA_TYPE_FLOAT16, Ah + total, 3, dims, strides, box,
                       CU_TENSOR_MAP_SWIZZLE_128B));
  }
  {
    const cuuint64_t dims[2] = {(cuuint64_t)G, (cuuint64_t)NT};
    const cuuint64_t strides[1] = {(cuuint64_t)G * 2};
    const cuuint32_t box[2] = {hc::BK, (cuuint32_t)NT};
    GM_TRY(encode_tmap(&tmBh, CU_TENSOR_MAP_DATA_TYPE_FLOAT16, Bh, 2, dims, strides, box, CU_TENSOR_MAP_SWIZZLE_64B));
    GM_TRY(encode_tmap(&tmBl, CU_TENSOR_MAP_DATA_TYPE_FLOAT16, Bl, 2, dims, strides, box, CU_TENSOR_MAP_SWIZZLE_64B));
  }
  hc::Params prm = {};
  prm.U = Ug; prm.Zh = nullptr; prm.u_plane_stride = (long long)Q * Npad;
  prm.rscale = rscale; prm.vbound = vbound; prm.bound_gain = 1.f; prm.zgain = 0.f;
  prm.Q = Q; prm.N = Npad; prm.NT = NT; prm.KB = KB; prm.n_rt = 1;
  prm.t_tiles = 1;
  prm.total_tiles = 1;
  prm.plane0 = 0; prm.stages = stages; prm.kchunk = 4;
  GM_TRY(ensure_dyn_smem(dev, (const void*)hc::k_contract_h<false>, hc::smem_bytes(NT, stages)));
  cudaLaunchConfig_t cfg = {};
  cfg.gridDim = dim3(1);
  cfg.blockDim = dim3(hc::NTHREADS);
  cfg.dynamicSmemBytes = hc::smem_bytes(NT, stages);
  cfg.stream = stream;
  GM_CUDA(cudaLaunchKernelEx(&cfg, hc::k_contract_h<false>, tmAh, tmAl, tmBh, tmBl, prm));
  k_expand_gram<<<(P * P * P * P + 255) / 256, 256, 0, stream>>>(Ug, Npad, P, dA, S_dev);
  GM_CUDA(cudaGetLastError());
  return 0;
}

}  // namespace

// ============================================================================================
extern "C" {

int gmmnlse_abi_version(void) { return 4; }

int gmmnlse_overlap_tensor(int P, long long G, const double* F, double dA, double* S_out) {
  if (P < 1 || G < 1 || !F || !S_out || !(dA > 0)) return GMMNLSE_EINVAL;
  if (G % hc::BK != 0) return GMMNLSE_EUNSUPPORTED;
  for (long long i = 0; i < (long long)P * G; ++i)
    if (!std::isfinite(F[i])) return GMMNLSE_EINVAL;
  return overlap_tensor_gpu(P, G, F, dA, S_out);
}

const char* gmmnlse_last_cuda_error(void) { return g_cuda_err.c_str(); }

const char* gmmnlse_status_string(int s) {
  switch (s) {
    case GMMNLSE_OK: return "ok";
    case GMMNLSE_WARN_NOCONV: return "warning: an MPA large step did not converge within max_iter";
    case GMMNLSE_EINVAL: return "invalid argument";
    case GMMNLSE_ENOMEM: return "out of memory";
    case GMMNLSE_ECUDA: return "CUDA error";
    case GMMNLSE_EUNSUPPORTED: return "unsupported configuration";
  }
  return "unknown status";
}

static int create_plan(gmmnlse_plan** out, int P, int N, int M, double dt, double dz, const double* beta,
                       int n_beta, const double* S, const double* S_R, bool general, bool tensors_complex,
                       double f_R, const double* h_R, double omega0, double n2, const gmmnlse_options* opt) {
  if (!out) return GMMNLSE_EINVAL;
  *out = nullptr;
  gmmnlse_options o = {0, 1, 1e-6, 0, 0, 0, 0, 0, 0, 0};
  if (opt) o = *opt;
  if (P < 1 || N < 1 || M < 1 || n_beta < 1 || !beta || !S) return GMMNLSE_EINVAL;
  if (N & (N - 1)) return GMMNLSE_EINVAL;
  if (!(dt > 0) || !(dz > 0) || !(omega0 > 0) || !std::isfinite(n2)) return GMMNLSE_EINVAL;
  if (!(f_R >= 0.0 && f_R <= 1.0)) return GMMNLSE_EINVAL;      // a fraction; the fp16 range bound assumes it
  if ((f_R != 0.0) != (h_R != nullptr)) return GMMNLSE_EINVAL;
  if (o.precision != 0 && o.precision != 1) return GMMNLSE_EINVAL;
  if (o.raman < 0 || o.raman > 2) return GMMNLSE_EINVAL;
  if (o.contraction != 0 && o.contraction != 1 && o.contraction != 3 && (o.contraction < 6 || o.contraction > 9))
    return GMMNLSE_EINVAL;
  if (o.graph < 0 || o.graph > 1) return GMMNLSE_EINVAL;
  if (o.stop_rule < 0 || o.stop_rule > 1) return GMMNLSE_EINVAL;
  if (o.async_call < 0 || o.async_call > 1) return GMMNLSE_EINVAL;
  if (o.shock && M_PI / dt >= omega0) return GMMNLSE_EINVAL;
  if (!(o.tol > 0)) o.tol = 1e-6;
  for (long long i = 0; i < (long long)P * n_beta; ++i)
    if (!std::isfinite(beta[i])) return GMMNLSE_EINVAL;
  if (general && !S_R) return GMMNLSE_EINVAL;
  const long long P4 = (long long)P * P * P * P * (general && tensors_complex ? 2 : 1);
  double smax = 0;
  for (long long i = 0; i < P4; ++i) {
    if (!std::isfinite(S[i]) || (general && !std::isfinite(S_R[i]))) return GMMNLSE_EINVAL;
    smax = std::fmax(smax, std::fabs(S[i]));
  }
  if (h_R)
    for (int i = 0; i < N; ++i)
      if (!std::isfinite(h_R[i])) return GMMNLSE_EINVAL;
  if (N < 16 || N > (o.precision ? 8192 : 16384)) return GMMNLSE_EUNSUPPORTED;
  // the packed-pair path needs S symmetric under m<->n and p<->l (Eq. 2 gives all 24 permutations)
  for (int p = 0; p < (general ? 0 : P); ++p)
    for (int l = 0; l < P; ++l)
      for (int m = 0; m < P; ++m)
        for (int n = 0; n < P; ++n) {
          const double a = S[(((size_t)p * P + l) * P + m) * P + n];
          const double b = S[(((size_t)p * P + l) * P + n) * P + m];
          const double c = S[(((size_t)l * P + p) * P + m) * P + n];
          if (std::fabs(a - b) > 1e-12 * smax || std::fabs(a - c) > 1e-12 * smax) return GMMNLSE_EUNSUPPORTED;
        }
  gmmnlse_plan* pl = nullptr;
  if (o.precision == 0) pl = new (std::nothrow) PlanT<float>();
  else pl = new (std::nothrow) PlanT<double>();
  if (!pl) return GMMNLSE_ENOMEM;
  pl->P = P; pl->N = N; pl->M = M; pl->log2N = ilog2(N); pl->precision = o.precision; pl->shock = o.shock ? 1 : 0;
  pl->dt = dt; pl->dz = dz; pl->f_R = f_R; pl->omega0 = omega0; pl->n2 = n2; pl->tol = o.tol;
  pl->max_iter = o.max_iter > 0 ? o.max_iter : 2 * M + 4;
  pl->fixed_iter = o.fixed_iter > 0 ? o.fixed_iter : 0;
  pl->contraction = o.contraction;
  pl->raman = o.raman;
  pl->graph = o.graph;
  pl->stop_rule = o.stop_rule;
  pl->async_call = o.async_call;
  if (cudaGetDevice(&pl->device) != cudaSuccess) { delete pl; g_cuda_err = "cudaGetDevice failed"; return GMMNLSE_ECUDA; }
  pl->general = general;
  pl->gen_complex = general && tensors_complex;
  pl->gen_SR = S_R;
  // Im D_w^(p) = beta0 + beta1 w + sum_{k>=2} beta_k w^k / k!
  pl->phi.assign((size_t)P * N, 0.0);
  for (int p = 0; p < P; ++p)
    for (int k = 0; k < N; ++k) {
      const double w = 2.0 * M_PI * (double)(k < N / 2 ? k : k - N) / (N * dt);
      double acc = 0, wp = 1, fact = 1;
      for (int b = 0; b < n_beta; ++b) {
        if (b > 0) { wp *= w; fact *= (double)b; }
        acc += beta[(size_t)p * n_beta + b] * wp / fact;
      }
      pl->phi[(size_t)p * N + k] = acc;
    }
  const int st = pl->init(S, h_R);
  pl->gen_SR = nullptr;
  if (st < 0) { delete pl; return st; }
  *out = pl;
  return GMMNLSE_OK;
}

int gmmnlse_plan_create(gmmnlse_plan** out, int P, int N, int M, double dt, double dz, const double* beta,
                        int n_beta, const double* S, double f_R, const double* h_R, double omega0, double n2,
                        const gmmnlse_options* opt) {
  return create_plan(out, P, N, M, dt, dz, beta, n_beta, S, nullptr, false, false, f_R, h_R, omega0, n2, opt);
}

int gmmnlse_plan_create_general(gmmnlse_plan** out, int P, int N, int M, double dt, double dz, const double* beta,
                                int n_beta, const double* S_K, const double* S_R, int tensors_complex, double f_R,
                                const double* h_R, double omega0, double n2, const gmmnlse_options* opt) {
  return create_plan(out, P, N, M, dt, dz, beta, n_beta, S_K, S_R, true, tensors_complex != 0, f_R, h_R, omega0, n2,
                     opt);
}

namespace {
struct StreamForCall {          // a non-NULL `stream` argument applies to this call only
  gmmnlse_plan* plan;
  cudaStream_t saved;
  StreamForCall(gmmnlse_plan* p, void* s) : plan(p), saved(p->stream) {
    if (s) p->stream = (cudaStream_t)s;
  }
  ~StreamForCall() { plan->stream = saved; }
};
}  // namespace

int gmmnlse_overlap_tensor_noalloc(int P, long long G, const double* F_dev, double dA, double* S_dev, void* stream) {
  if (P < 1 || G < 1 || !F_dev || !S_dev || !(dA > 0)) return GMMNLSE_EINVAL;
  if (P > NOALLOC_PMAX || G > NOALLOC_GMAX) {
    g_cuda_err = "gmmnlse_overlap_tensor_noalloc: P = " + std::to_string(P) + ", G = " + std::to_string(G) +
                 " exceed the static scratch (P <= " + std::to_string(NOALLOC_PMAX) + ", G <= " +
                 std::to_string(NOALLOC_GMAX) + "); use gmmnlse_overlap_tensor";
    return GMMNLSE_EUNSUPPORTED;
  }
  if (G % hc::BK != 0) {
    g_cuda_err = "gmmnlse_overlap_tensor_noalloc: G must be a multiple of 32";
    return GMMNLSE_EUNSUPPORTED;
  }
  return overlap_tensor_noalloc(P, G, F_dev, dA, S_dev, (cudaStream_t)stream);
}

int gmmnlse_overlap_tensor_noalloc_limits(int* P_max, long long* G_max, long long* scratch_bytes) {
  if (P_max) *P_max = NOALLOC_PMAX;
  if (G_max) *G_max = NOALLOC_GMAX;
  if (scratch_bytes) *scratch_bytes = (long long)NOALLOC_BYTES;
  return GMMNLSE_OK;
}

int gmmnlse_propagate(gmmnlse_plan* plan, const void* A_in, double L, void* A_out, void* stream) {
  if (!plan || !A_in || !A_out) return GMMNLSE_EINVAL;
  DeviceGuard dg(plan->device);
  StreamForCall sc(plan, stream);
  return plan->propagate(A_in, L, A_out);
}

int gmmnlse_propagate_host(gmmnlse_plan* plan, const void* A_in_host, double L, void* A_out_host) {
  if (!plan || !A_in_host || !A_out_host) return GMMNLSE_EINVAL;
  const double ns = L / plan->dz;
  if (!(L >= 0) || std::fabs(ns - std::round(ns)) > 1e-9 * std::fmax(1.0, ns)) return GMMNLSE_EINVAL;
  DeviceGuard dg(plan->device);
  return plan->propagate_host(A_in_host, L, A_out_host);
}

int gmmnlse_propagate_rk4ip(gmmnlse_plan* plan, const void* A_in, double L, void* A_out, void* stream) {
  if (!plan || !A_in || !A_out) return GMMNLSE_EINVAL;
  DeviceGuard dg(plan->device);
  StreamForCall sc(plan, stream);
  return plan->propagate_rk4ip(A_in, L, A_out);
}

int gmmnlse_set_gain(gmmnlse_plan* plan, const double* g) {
  if (!plan) return GMMNLSE_EINVAL;
  DeviceGuard dg(plan->device);
  return plan->set_gain(g);
}

int gmmnlse_set_coupling(gmmnlse_plan* plan, const double* Q) {
  if (!plan) return GMMNLSE_EINVAL;
  DeviceGuard dg(plan->device);
  return plan->set_coupling(Q);
}

int gmmnlse_set_coupling_profile(gmmnlse_plan* plan, const double* f, int n) {
  if (!plan) return GMMNLSE_EINVAL;
  DeviceGuard dg(plan->device);
  return plan->set_coupling_profile(f, n);
}

int gmmnlse_set_gain_saturation(gmmnlse_plan* plan, double g_sat) {
  if (!plan) return GMMNLSE_EINVAL;
  DeviceGuard dg(plan->device);
  return plan->set_gain_saturation(g_sat);
}

int gmmnlse_shard_begin(gmmnlse_plan* plan, const void* A_in) {
  if (!plan || !A_in) return GMMNLSE_EINVAL;
  DeviceGuard dg(plan->device);
  return plan->shard_begin(A_in);
}

int gmmnlse_shard_iterate(gmmnlse_plan* plan, int j_lo, int j_hi, int Mc, int first, void* block_sum) {
  if (!plan || !block_sum) return GMMNLSE_EINVAL;
  DeviceGuard dg(plan->device);
  return plan->shard_iterate(j_lo, j_hi, Mc, first, block_sum);
}

int gmmnlse_shard_update(gmmnlse_plan* plan, int j_lo, int j_hi, int Mc, int first, const void* all_sums, int shard,
                         int n_shards, double* err_local) {
  if (!plan || !all_sums) return GMMNLSE_EINVAL;
  DeviceGuard dg(plan->device);
  return plan->shard_update(j_lo, j_hi, Mc, first, all_sums, shard, n_shards, err_local);
}

int gmmnlse_shard_advance(gmmnlse_plan* plan, int Mc, const void* all_sums, int n_shards) {
  if (!plan || !all_sums) return GMMNLSE_EINVAL;
  DeviceGuard dg(plan->device);
  return plan->shard_advance(Mc, all_sums, n_shards);
}

int gmmnlse_shard_end(gmmnlse_plan* plan, void* A_out) {
  if (!plan || !A_out) return GMMNLSE_EINVAL;
  DeviceGuard dg(plan->device);
  return plan->shard_end(A_out);
}

int gmmnlse_nonlinear_op(gmmnlse_plan* plan, const void* A, void* dA) {
  if (!plan || !A || !dA || A == dA) return GMMNLSE_EINVAL;
  DeviceGuard dg(plan->device);
  return plan->nonlinear_op(A, dA);
}

int gmmnlse_set_stream(gmmnlse_plan* plan, void* stream) {
  if (!plan) return GMMNLSE_EINVAL;
  plan->stream = (cudaStream_t)stream;
  return GMMNLSE_OK;
}

int gmmnlse_get_stats(const gmmnlse_plan* plan, long long* large_steps, long long* iterations, double* last_err,
                      long long* not_converged) {
  if (!plan) return GMMNLSE_EINVAL;
  {                                                  // options.async_call: the last call's counters may still be in flight
    DeviceGuard dg(plan->device);
    GM_TRY(const_cast<gmmnlse_plan*>(plan)->fold_pending());
  }
  if (large_steps) *large_steps = plan->n_large;
  if (iterations) *iterations = plan->n_iter;
  if (last_err) *last_err = plan->last_err;
  if (not_converged) *not_converged = plan->n_noconv;
  return GMMNLSE_OK;
}

long long gmmnlse_launch_count(const gmmnlse_plan* plan) {
  if (!plan) return 0;
  DeviceGuard dg(plan->device);
  const_cast<gmmnlse_plan*>(plan)->fold_pending();
  return plan->n_launch;
}

int gmmnlse_profile_enable(gmmnlse_plan* plan, int on) {
  if (!plan) return GMMNLSE_EINVAL;
  DeviceGuard dg(plan->device);
  if (plan->prof_collect() < 0) return GMMNLSE_ECUDA;
  plan->prof_on = on != 0;
  if (on)
    for (int k = 0; k < GMMNLSE_KIND_COUNT; ++k) { plan->prof_ms[k] = 0; plan->prof_n[k] = 0; }
  return GMMNLSE_OK;
}

int gmmnlse_profile_get(gmmnlse_plan* plan, int kind, double* total_ms, long long* launches) {
  if (!plan || kind < 0 || kind >= GMMNLSE_KIND_COUNT) return GMMNLSE_EINVAL;
  DeviceGuard dg(plan->device);
  if (plan->prof_collect() < 0) return GMMNLSE_ECUDA;
  if (total_ms) *total_ms = plan->prof_ms[kind];
  if (launches) *launches = plan->prof_n[kind];
  return GMMNLSE_OK;
}

int gmmnlse_debug_get_planes(gmmnlse_plan* plan, void* out_host) {
  if (!plan || !out_host) return GMMNLSE_EINVAL;
  DeviceGuard dg(plan->device);
  return plan->get_planes(out_host);
}

int gmmnlse_debug_fft(gmmnlse_plan* plan, const void* in, void* out, int rows, int dir) {
  if (!plan || !in || !out) return GMMNLSE_EINVAL;
  DeviceGuard dg(plan->device);
  return plan->debug_fft(in, out, rows, dir);
}

int gmmnlse_debug_pairs(gmmnlse_plan* plan, const void* A, void* V, int n_planes) {
  if (!plan || !A || !V) return GMMNLSE_EINVAL;
  DeviceGuard dg(plan->device);
  return plan->debug_pairs(A, V, n_planes);
}

int gmmnlse_debug_contract(gmmnlse_plan* plan, const void* V, void* U, int n_planes) {
  if (!plan || !V || !U || V == U) return GMMNLSE_EINVAL;
  DeviceGuard dg(plan->device);
  return plan->debug_contract(V, U, n_planes);
}

int gmmnlse_contraction_kind(const gmmnlse_plan* plan) { return plan ? plan->contraction_kind() : 0; }

int gmmnlse_raman_kind(const gmmnlse_plan* plan) { return plan ? plan->raman_kind() : 0; }

int gmmnlse_lowrank_rank(const gmmnlse_plan* plan) { return plan ? plan->lowrank_rank() : 0; }

int gmmnlse_sparse_info(const gmmnlse_plan* plan, int* classes, double* work_fraction) {
  return plan ? plan->sparse_info(classes, work_fraction) : GMMNLSE_EINVAL;
}

int gmmnlse_loop_kind(const gmmnlse_plan* plan) { return plan ? plan->loop_state : 0; }

int gmmnlse_debug_set_tc_chunk(gmmnlse_plan* plan, int k) {
  if (!plan) return GMMNLSE_EINVAL;
  DeviceGuard dg(plan->device);
  return plan->set_tc_chunk(k);
}

void gmmnlse_plan_destroy(gmmnlse_plan* plan) {
  if (!plan) return;
  DeviceGuard dg(plan->device);
  delete plan;
}

}  // extern "C"
