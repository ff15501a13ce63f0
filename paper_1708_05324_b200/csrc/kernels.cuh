// CUDA kernels of the MPA hot path.  Templated on the real type
// T (float: complex64 path, double: complex128 path) and on log2 N.
#pragma once
#include "fft.cuh"
#include "gemm_h.cuh"
#include "ptx_sm100.cuh"

namespace gm {

// ------------------------------------------------------------------------------------------
// a1 / a3 / a8 / a12: row FFT with fused pre- and post-multiplies.
//   grid = (P, n_planes); row (j, p) = in + j*in_plane_stride + p*N   (in_plane_stride may be 0:
//   every plane reads psi_0 -- the first MPA iterate)
//   x_n   = in[n] * (pre ? pre[j][p][n] : 1)                      Eq. 11: psi_j * exp(+D j dz)
//   X_k   = FFT_DIR(x)
//   out_k = X_k * scale * (post_vec ? post_vec[k] : 1) * (post_tab ? conj(post_tab[j][p][k]) : 1)
//                                                        Eq. 12: K(w) exp(-D j dz) F{N_p}
//   bound (optional; zeroed before the launch): bound[0] = max(bound[0], bound_gain max |out|^2) -- the range bound of
//   the fp16 pair streams that k_bound_field would otherwise recompute from the stored planes (a3 of the MPA iteration).
template <typename T, int LOG2N, int DIR>
__global__ void __launch_bounds__((1 << LOG2N) / 16, ((1 << LOG2N) / 16 == 512 && sizeof(T) == 4) ? 2 : 1)
k_fft_rows(const cplx<T>* __restrict__ in, long long in_plane_stride, cplx<T>* __restrict__ out,
           long long out_plane_stride, const cplx<T>* __restrict__ pre, const cplx<T>* __restrict__ post_vec,
           const cplx<T>* __restrict__ post_tab, long long tab_plane_stride, T scale,
           const cplx<T>* __restrict__ tw, const T* __restrict__ row_scale, float* __restrict__ bound, float bound_gain) {
  pdl_prologue();
  constexpr int N = 1 << LOG2N;
  extern __shared__ __align__(16) unsigned char smem_raw[];
  cplx<T>* sm = reinterpret_cast<cplx<T>*>(smem_raw);
  const int p = blockIdx.x, j = blockIdx.y;
  const cplx<T>* src = in + j * in_plane_stride + (long long)p * N;
  cplx<T>* dst = out + j * out_plane_stride + (long long)p * N;
  const long long toff = j * tab_plane_stride + (long long)p * N;
  const cplx<T>* pre_r = pre ? pre + toff : nullptr;
  const cplx<T>* post_r = post_tab ? post_tab + toff : nullptr;
  if (row_scale) scale *= row_scale[j * gridDim.x + p];     // gain: exp(+-g_p j dz), one factor per (plane, mode)
  float amax = 0.f;
  block_fft<T, LOG2N, DIR>(
      sm, tw,
      [&](int n) {
        cplx<T> x = src[n];
        if (pre_r) x = cmul(x, pre_r[n]);
        return x;
      },
      [&](int k, cplx<T> X) {
        X = cscale(X, scale);
        if (post_vec) X = cmul(X, post_vec[k]);
        if (post_r) X = cmulc(X, post_r[k]);
        dst[k] = X;
        if (bound) amax = fmaxf(amax, (float)(X.x * X.x + X.y * X.y));
      });
  if (bound) {                                              // uniform branch: one atomic per warp
#pragma unroll
    for (int d = 16; d > 0; d >>= 1) amax = fmaxf(amax, __shfl_xor_sync(0xffffffffu, amax, d));
    if ((threadIdx.x & 31) == 0 && amax > 0.f) atomicMax(reinterpret_cast<unsigned int*>(bound), __float_as_uint(amax * bound_gain));
  }
}

// fp16 split output of the pair kernels for the kind::f16 contraction (gemm_h.cuh): V' = sV V as Vh + Vl, two
// fp16 arrays per plane ([Q][N] hi rows, then [Q][N] lo rows: the bytes of the fp32 V plane they replace).
// sV = hc::v_scale(*vbound): a power of two that puts the launch's largest |V| below 2^14.  Vh == nullptr: fp32 V.
struct HalfOut {
  __half* Vh;
  long long plane_stride;      // halves between planes (2 Q N)
  long long lo_offset;         // halves from a hi row to its lo row (Q N)
  int N;
  const float* vbound;
  const int* vrow;             // block-sparse form: stream q is stored at row vrow[q] (class order); null = row q
  __device__ __forceinline__ long long row(long long q) const { return vrow ? (long long)vrow[q] : q; }
  __device__ __forceinline__ void store(int j, int q, int n, float v) const {
    const float x = v * hc::v_scale(*vbound, false);
    const __half h = __float2half_rn(x);
    __half* d = Vh + j * plane_stride + row(q) * N + n;
    d[0] = h;
    d[lo_offset] = __float2half_rn(x - __half2float(h));
  }
};

// bound[0] = max(bound[0], gain * max |A|^2) over `planes` planes of n complex samples (bound zeroed before the
// launch; non-negative floats order like their bit patterns).  |Re / Im (A_m A_n*)| <= max |A|^2, and `gain`
// bounds the instantaneous + Raman-convolved weights of a stream, so bound >= every |V| the pair kernel writes.
template <typename T>
__global__ void __launch_bounds__(256)
k_bound_field(const cplx<T>* __restrict__ A, long long a_plane_stride, long long n, float gain, float* bound) {
  pdl_prologue();
  const cplx<T>* a = A + blockIdx.y * a_plane_stride;
  float m = 0.f;
  for (long long i = (long long)blockIdx.x * 256 + threadIdx.x; i < n; i += (long long)gridDim.x * 256) {
    const cplx<T> v = a[i];
    m = fmaxf(m, (float)(v.x * v.x + v.y * v.y));
  }
#pragma unroll
  for (int d = 16; d > 0; d >>= 1) m = fmaxf(m, __shfl_xor_sync(0xffffffffu, m, d));
  if ((threadIdx.x & 31) == 0 && m > 0.f) atomicMax(reinterpret_cast<unsigned int*>(bound), __float_as_uint(m * gain));
}
// same for an array of n real samples: bound[0] = max(bound[0], max |V|)
template <typename T>
__global__ void __launch_bounds__(256)
k_bound_real(const T* __restrict__ V, long long n, float* bound) {
  pdl_prologue();
  float m = 0.f;
  for (long long i = (long long)blockIdx.x * 256 + threadIdx.x; i < n; i += (long long)gridDim.x * 256)
    m = fmaxf(m, fabsf((float)V[i]));
#pragma unroll
  for (int d = 16; d > 0; d >>= 1) m = fmaxf(m, __shfl_xor_sync(0xffffffffu, m, d));
  if ((threadIdx.x & 31) == 0 && m > 0.f) atomicMax(reinterpret_cast<unsigned int*>(bound), __float_as_uint(m * 1.0001f));
}

// fp32 V[planes][Q][N] -> fp16 split planes (for a caller-supplied V: gmmnlse_debug_contract)
__global__ void __launch_bounds__(256)
k_v_encode(const float* __restrict__ Vin, long long QN, long long total, HalfOut ho) {
  pdl_prologue();
  for (long long i = (long long)blockIdx.x * 256 + threadIdx.x; i < total; i += (long long)gridDim.x * 256) {
    const int j = (int)(i / QN);
    const long long r = i - j * QN;
    ho.store(j, (int)(r / ho.N), (int)(r % ho.N), Vin[i]);
  }
}

// Per-stream description of the general form of Eq. 1 (S^K != S^R, complex, no symmetry; NEXT-2): stream q is
// Re (kind 0) or Im (kind 1) of A_m A_n*, weighted wk[q] on its instantaneous part and wr[q] on its Raman-
// convolved part.  All-null = the scalar-mode path (every stream Re, weights folded into H / cs, omf).
// The two streams of one CTA (q0 = 2 bx, q0 + 1) always share their weights (blocks are padded to even size).
template <typename T> struct StreamSpec {
  const int* kind;
  const T* wk;
  const T* wr;
};
template <typename C>
__device__ __forceinline__ auto pair_stream(C a, C b, bool imag) -> decltype(a.x) {
  return imag ? a.y * b.x - a.x * b.y : a.x * b.x + a.y * b.y;       // Im / Re of a b*
}

// ------------------------------------------------------------------------------------------
// a4 + a5: pair products and Raman convolution, two real pair streams per complex FFT.
//   grid = (ceil(Q/2), n_planes).  CTA (qq, j) handles packed pairs q0 = 2 qq, q1 = q0 + 1:
//   z_n = Re(A_m A_n*)[q0] + i Re(A_m A_n*)[q1];  Z = F{z};  Z *= H,  H = ((1-fR) + fR ht_R)/N;
//   v = F^-1{Z};  V[q0] = Re v, V[q1] = Im v.        (Eq. 1 bracket; h_R real)
// With HAS_RAMAN == false the FFTs are skipped: V = Re T.
template <typename T, int LOG2N, bool HAS_RAMAN>
__global__ void __launch_bounds__((1 << LOG2N) / 16)
k_pair_conv(const cplx<T>* __restrict__ A, long long a_plane_stride, T* __restrict__ V, long long v_plane_stride,
            const int* __restrict__ pair_m, const int* __restrict__ pair_n, int Q,
            const cplx<T>* __restrict__ H, const cplx<T>* __restrict__ tw, StreamSpec<T> gs, HalfOut ho) {
  pdl_prologue();
  constexpr int N = 1 << LOG2N, NT = N / 16;
  extern __shared__ __align__(16) unsigned char smem_raw[];
  cplx<T>* sm = reinterpret_cast<cplx<T>*>(smem_raw);
  const int q0 = 2 * blockIdx.x, q1 = q0 + 1, j = blockIdx.y;
  const bool has1 = q1 < Q;
  {
    // phase 1: z_n = Re(A_m A_n*)[q0] + i Re(A_m A_n*)[q1], formed straight from the four field rows.  Kept
    // apart from the FFT so that its pointers and in-flight loads do not add to the FFT's register peak
    // (N = 16384 runs 1024 threads, i.e. 64 registers per thread).
    const cplx<T>* Aj = A + j * a_plane_stride;
    const cplx<T>* am0 = Aj + (long long)pair_m[q0] * N;
    const cplx<T>* an0 = Aj + (long long)pair_n[q0] * N;
    const cplx<T>* am1 = Aj + (long long)pair_m[has1 ? q1 : q0] * N;
    const cplx<T>* an1 = Aj + (long long)pair_n[has1 ? q1 : q0] * N;
    T* v0 = V + j * v_plane_stride + (long long)q0 * N;
    T* v1 = V + j * v_plane_stride + (long long)q1 * N;
    const bool im0 = gs.kind && gs.kind[q0], im1 = gs.kind && has1 && gs.kind[q1];
    const T wk = gs.wk ? gs.wk[q0] : (T)1;
#pragma unroll 4
    for (int e = 0; e < 16; ++e) {
      const int n = threadIdx.x + e * NT;
      const cplx<T> a = am0[n], b = an0[n], c = am1[n], d = an1[n];
      const cplx<T> z = mk(pair_stream(a, b, im0), has1 ? pair_stream(c, d, im1) : (T)0);
      if constexpr (HAS_RAMAN) {
        sm[fft_pad(n)] = z;
      } else if (ho.Vh) {
        ho.store(j, q0, n, (float)(wk * z.x));
        if (has1) ho.store(j, q1, n, (float)(wk * z.y));
      } else {
        v0[n] = wk * z.x;
        if (has1) v1[n] = wk * z.y;
      }
    }
  }
  if constexpr (HAS_RAMAN) {
    __syncthreads();
    // phase 2: Z = F{z} . H   (H = ((1-fR) + fR ht_R)/N; general streams: H_q = wk_q/N + wr_q ht_R/N), in place
    const T wkN = gs.wk ? gs.wk[q0] / (T)N : (T)0, wr = gs.wr ? gs.wr[q0] : (T)0;
    block_fft<T, LOG2N, +1>(sm, tw, [&](int n) { return sm[fft_pad(n)]; },
                            [&](int k, cplx<T> Z) {
                              cplx<T> h = H[k];
                              if (gs.wk) h = mk(wkN + wr * h.x, wr * h.y);     // H holds ht_R/N in general mode
                              sm[fft_pad(k)] = cmul(Z, h);
                            });
    __syncthreads();
    // phase 3: v = F^-1{Z};  V[q0] = Re v, V[q1] = Im v
    T* v0 = V + j * v_plane_stride + (long long)q0 * N;
    block_fft<T, LOG2N, -1>(
        sm, tw, [&](int k) { return sm[fft_pad(k)]; },
        [&](int n, cplx<T> v) {
          if (ho.Vh) {
            ho.store(j, q0, n, (float)v.x);
            if (has1) ho.store(j, q1, n, (float)v.y);
          } else {
            v0[n] = v.x;
            if (has1) v0[N + n] = v.y;
          }
        });
  }
}

// ------------------------------------------------------------------------------------------
// a4 + a5, recursive form.  When the sampled response is a damped oscillation, h_R[j] = Im(c zeta^j) (the
// form BASELINE.json's tau1, tau2 give; detected at plan time from the samples themselves), the circular
// convolution of Eq. 1 is a one-pole complex recurrence along t,
//   w[i] = x[i] + zeta w[i-1],   (h_R (*) x)[i] = dt Im(c w[i]),
// exact up to zeta^N (< 1e-14, checked).  Each thread owns 16 consecutive samples of two pair streams; chunk
// carries are combined by a warp-shuffle scan of the recurrence (multipliers zeta^(16 d) from the table
// zp[m] = zeta^(16 m)), warp totals through shared memory, and the periodic wrap w[-1] = w[N-1] closes the
// circle.  No FFT: the kernel is one read of the field rows and one write of V.
//   cs = c dt f_R,  omf = 1 - f_R;  V = omf x + Im(cs w).
template <typename T, int LOG2N, bool GEN>
__global__ void __launch_bounds__((1 << LOG2N) / 16)
k_pair_iir(const cplx<T>* __restrict__ A, long long a_plane_stride, T* __restrict__ V, long long v_plane_stride,
           const int* __restrict__ pair_m, const int* __restrict__ pair_n, int Q, cplx<T> zeta, cplx<T> cs, T omf,
           const cplx<T>* __restrict__ zp, StreamSpec<T> gs, HalfOut ho) {
  pdl_prologue();
  constexpr int N = 1 << LOG2N, NT = N / 16, NW = (NT + 31) / 32;
  extern __shared__ __align__(16) unsigned char smem_raw[];
  cplx<T>* sm = reinterpret_cast<cplx<T>*>(smem_raw);         // fft_smem_elems(N) + 2 * (NW + 1) complex
  cplx<T>* wt = sm + fft_smem_elems(N);                       // [2][NW] warp totals, then [2] row totals
  const int q0 = 2 * blockIdx.x, q1 = q0 + 1, j = blockIdx.y, tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  const bool has1 = q1 < Q;
  {
    const cplx<T>* Aj = A + j * a_plane_stride;
    const cplx<T>* am0 = Aj + (long long)pair_m[q0] * N;
    const cplx<T>* an0 = Aj + (long long)pair_n[q0] * N;
    const cplx<T>* am1 = Aj + (long long)pair_m[has1 ? q1 : q0] * N;
    const cplx<T>* an1 = Aj + (long long)pair_n[has1 ? q1 : q0] * N;
    const bool im0 = GEN && gs.kind[q0], im1 = GEN && has1 && gs.kind[q1];
    // consecutive packed pairs (m, n), (m, n + 1) share row m except across a row end: read it once (the kernel is
    // bound by L1 throughput, and a quarter of its global loads were this second read)
    const bool same_m = am1 == am0;
#pragma unroll 4
    for (int e = 0; e < 16; ++e) {
      const int n = tid + e * NT;
      const cplx<T> a = am0[n], b = an0[n], d = an1[n];
      const cplx<T> c = same_m ? a : am1[n];
      sm[fft_pad(n)] = mk(pair_stream(a, b, im0), has1 ? pair_stream(c, d, im1) : (T)0);
    }
  }
  if constexpr (GEN) {                                        // general streams: per-stream Kerr / Raman weights
    omf = gs.wk[q0];
    cs = cscale(cs, gs.wr[q0]);
  }
  __syncthreads();
  cplx<T> x[16];                                              // x.x: stream q0, x.y: stream q1; samples 16 tid + e
#pragma unroll
  for (int e = 0; e < 16; ++e) x[e] = sm[17 * tid + e];       // fft_pad(16 k + e) = 17 k + e: conflict-free
  cplx<T> w0 = mk((T)0, (T)0), w1 = w0;
#pragma unroll
  for (int e = 0; e < 16; ++e) {
    w0 = mk(x[e].x + zeta.x * w0.x - zeta.y * w0.y, zeta.x * w0.y + zeta.y * w0.x);
    w1 = mk(x[e].y + zeta.x * w1.x - zeta.y * w1.y, zeta.x * w1.y + zeta.y * w1.x);
  }
  // inclusive scan of the chunk totals inside the warp: T_k = sum_{i<=k} zeta^(16 (k-i)) E_i
  const unsigned mask = NT >= 32 ? 0xffffffffu : ((1u << NT) - 1u);
#pragma unroll
  for (int d = 1; d < 32 && d < NT; d <<= 1) {
    const cplx<T> p = zp[d];
    const T r0x = __shfl_up_sync(mask, w0.x, d), r0y = __shfl_up_sync(mask, w0.y, d);
    const T r1x = __shfl_up_sync(mask, w1.x, d), r1y = __shfl_up_sync(mask, w1.y, d);
    if (lane >= d) {
      w0 = mk(w0.x + p.x * r0x - p.y * r0y, w0.y + p.x * r0y + p.y * r0x);
      w1 = mk(w1.x + p.x * r1x - p.y * r1y, w1.y + p.x * r1y + p.y * r1x);
    }
  }
  if (lane == 31 || tid == NT - 1) { wt[warp] = w0; wt[NW + warp] = w1; }
  // exclusive value inside the warp
  cplx<T> e0 = mk(__shfl_up_sync(mask, w0.x, 1), __shfl_up_sync(mask, w0.y, 1));
  cplx<T> e1 = mk(__shfl_up_sync(mask, w1.x, 1), __shfl_up_sync(mask, w1.y, 1));
  if (lane == 0) { e0 = mk((T)0, (T)0); e1 = e0; }
  __syncthreads();
  // carry into this warp's first chunk from the warps before it (zero history): zeta^512 per warp step
  cplx<T> g0 = mk((T)0, (T)0), g1 = g0;
  const cplx<T> z32 = zp[NT >= 32 ? 32 : NT];
  for (int i = 0; i < warp; ++i) {
    const cplx<T> a0 = wt[i], a1 = wt[NW + i];
    g0 = mk(a0.x + z32.x * g0.x - z32.y * g0.y, a0.y + z32.x * g0.y + z32.y * g0.x);
    g1 = mk(a1.x + z32.x * g1.x - z32.y * g1.y, a1.y + z32.x * g1.y + z32.y * g1.x);
  }
  if (tid == NT - 1) {                                        // row total with zero history = w[N-1] = w[-1]
    const cplx<T> pl = zp[lane + 1];
    wt[2 * NW] = mk(w0.x + pl.x * g0.x - pl.y * g0.y, w0.y + pl.x * g0.y + pl.y * g0.x);
    wt[2 * NW + 1] = mk(w1.x + pl.x * g1.x - pl.y * g1.y, w1.y + pl.x * g1.y + pl.y * g1.x);
  }
  __syncthreads();
  {
    const cplx<T> pl = zp[lane], pk = zp[tid], c0 = wt[2 * NW], c1 = wt[2 * NW + 1];
    // carry into chunk tid: exclusive in-warp part + zeta^(16 lane) warp carry + zeta^(16 tid) wrap-around
    w0 = mk(e0.x + pl.x * g0.x - pl.y * g0.y + pk.x * c0.x - pk.y * c0.y,
            e0.y + pl.x * g0.y + pl.y * g0.x + pk.x * c0.y + pk.y * c0.x);
    w1 = mk(e1.x + pl.x * g1.x - pl.y * g1.y + pk.x * c1.x - pk.y * c1.y,
            e1.y + pl.x * g1.y + pl.y * g1.x + pk.x * c1.y + pk.y * c1.x);
  }
#pragma unroll
  for (int e = 0; e < 16; ++e) {
    w0 = mk(x[e].x + zeta.x * w0.x - zeta.y * w0.y, zeta.x * w0.y + zeta.y * w0.x);
    w1 = mk(x[e].y + zeta.x * w1.x - zeta.y * w1.y, zeta.x * w1.y + zeta.y * w1.x);
    sm[17 * tid + e] = mk(omf * x[e].x + cs.x * w0.y + cs.y * w0.x, omf * x[e].y + cs.x * w1.y + cs.y * w1.x);
  }
  __syncthreads();
  if (ho.Vh) {                                                // fp16 hi / lo pairs, two samples per thread and store
    const float sv = hc::v_scale(*ho.vbound, false);
    __half2* h0 = reinterpret_cast<__half2*>(ho.Vh + j * ho.plane_stride + ho.row(q0) * N);
    __half2* l0 = reinterpret_cast<__half2*>(ho.Vh + j * ho.plane_stride + ho.lo_offset + ho.row(q0) * N);
    const long long d1 = has1 ? (ho.row(q1) - ho.row(q0)) * (N / 2) : 0;        // half2 units from row q0 to row q1
#pragma unroll 4
    for (int e = 0; e < 8; ++e) {
      const int n2 = tid + e * NT;                            // samples 2 n2, 2 n2 + 1
      const cplx<T> a = sm[fft_pad(2 * n2)], b = sm[fft_pad(2 * n2 + 1)];
      const float2 s0 = make_float2((float)a.x * sv, (float)b.x * sv), s1 = make_float2((float)a.y * sv, (float)b.y * sv);
      const __half2 hh0 = __float22half2_rn(s0), hh1 = __float22half2_rn(s1);
      const float2 f0 = __half22float2(hh0), f1 = __half22float2(hh1);
      h0[n2] = hh0;
      l0[n2] = __float22half2_rn(make_float2(s0.x - f0.x, s0.y - f0.y));
      if (has1) {
        h0[d1 + n2] = hh1;
        l0[d1 + n2] = __float22half2_rn(make_float2(s1.x - f1.x, s1.y - f1.y));
      }
    }
    return;
  }
  T* v0 = V + j * v_plane_stride + (long long)q0 * N;
#pragma unroll 4
  for (int e = 0; e < 16; ++e) {
    const int n = tid + e * NT;
    const cplx<T> v = sm[fft_pad(n)];
    v0[n] = v.x;
    if (has1) v0[N + n] = v.y;
  }
}

// ------------------------------------------------------------------------------------------
// a4 + a5, recursive form, register-blocked over mode rows (complex64, scalar-mode path).  The kernel above moves
// 1.75 field rows through L2 per pair stream and transposes every sample through shared memory twice; it is bound
// by L1/L2 throughput and latency, not by the HBM write of V.  Here a thread owns 16 CONSECUTIVE samples (128 B)
// of a row.  TMA brings each warp's 32 x 128 B slice of a field row into shared memory under the 128-byte swizzle
// (16-byte chunk c of thread t at slot c ^ (t & 7): conflict-free 128-bit reads, no transpose, no load
// instructions, no registers held across the latency); the rows m0, m0 + 1 of a CTA stay parked, the rows n of
// its range stream through one buffer that is refilled for n + 1 as soon as x = Re(A_m A_n*) has been formed:
// two streams (m0, n), (m0 + 1, n) per row load, 0.56-0.63 rows of L2 traffic per stream.  The recurrence
// w[i] = x[i] + zeta w[i-1] runs from a zero state per thread, chunk totals are combined by a warp-shuffle scan,
// and the carry into a warp's first chunk is the zero-history total of the warp before it (the last warp for
// warp 0: the periodic wrap): what that leaves out is zeta^512 of older history, < 1e-12 by the plan-time check
// that selects this kernel.  V leaves as 256-bit stores (32 contiguous bytes per lane, full sectors).
//   grid = (n_work, planes), block = N / 16; work[i] = (m0, n_begin, n_end): streams (m0, n), (m0 + 1, n), n in
//   [n_begin, n_end), m <= n only.  V row of (m, n): q = m P - m (m - 1) / 2 + (n - m).
//   tmA: field [planes][P][N/16][32 floats], box 32 x 32 x 1 x 1, SWIZZLE_128B; plane0 = first plane of the launch.
//   HALF_OUT: V as fp16 hi / lo rows scaled by v_scale(*vbound) (HalfOut), else fp32.
__device__ __forceinline__ void stg256(void* p, const uint32_t (&v)[8]) {
  asm volatile("st.global.v8.b32 [%0], {%1,%2,%3,%4,%5,%6,%7,%8};" ::"l"(p), "r"(v[0]), "r"(v[1]), "r"(v[2]),
               "r"(v[3]), "r"(v[4]), "r"(v[5]), "r"(v[6]), "r"(v[7]) : "memory");
}
struct PairWork { int m0, n_begin, n_end; };
struct ZetaPow { float re[16], im[16]; };                              // zeta^k, k = 0..15 (kernel argument: constant bank)

//   SEGS > 1 (N = 16384: three whole rows do not fit shared memory): a CTA handles one of SEGS segments of the row
//   plus a HALO warp in front of it (local warp 0 = the global warp before the segment, circularly).  The carry into a
//   warp's first chunk is the zero-history total of the warp before it, which depends on that warp's own 512 samples
//   only, so the halo warp recomputes it (first pass + scan) and writes nothing.  grid.x = n_work * SEGS.
template <int LOG2N, bool HALF_OUT, int SEGS = 1>
__global__ void __launch_bounds__((1 << LOG2N) / 16 / SEGS + (SEGS > 1 ? 32 : 0), 1)
k_pair_iir_rows(const __grid_constant__ CUtensorMap tmA, int plane0, float* __restrict__ V, long long v_plane_stride,
                int P, const PairWork* __restrict__ work, float2 zeta, float2 cs, float omf,
                const float2* __restrict__ zp, HalfOut ho, const ZetaPow zk) {
  pdl_prologue();
  using namespace ptx;
  constexpr bool HALO = SEGS > 1;
  constexpr int N = 1 << LOG2N, NWG = N / 512, NWM = NWG / SEGS;       // warps per row; main warps per CTA
  constexpr int NW = NWM + (HALO ? 1 : 0), NT = 32 * NW;               // local warps and threads (slices in shared memory)
  constexpr uint32_t ROW_BYTES = NT * 128, WARP_BYTES = 32 * 128;
  extern __shared__ unsigned char smem_raw[];
  const uint32_t raw_addr = smem_u32(smem_raw);
  const uint32_t base = (raw_addr + 1023u) & ~1023u;                  // swizzle atoms are 1 KiB
  unsigned char* sm = smem_raw + (base - raw_addr);
  const float4* rows = reinterpret_cast<const float4*>(sm);           // [0] m0, [1] m0 + 1, [2] streamed n
  float2* wt = reinterpret_cast<float2*>(sm + 3 * ROW_BYTES);         // [2 parity][NW][2 streams] warp totals
  const uint32_t bars = base + 3 * ROW_BYTES + 2 * NW * 2 * 8;        // [NW][2]: parked rows, streamed row
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5, j = blockIdx.y;
  const int seg = HALO ? (int)blockIdx.x % SEGS : 0;
  const PairWork wk = work[HALO ? blockIdx.x / SEGS : blockIdx.x];
  const bool halo_warp = HALO && warp == 0;
  // this warp's place in the row: global warp index and the first sample of this thread
  const int gw = HALO ? (seg * NWM + warp - 1 + NWG) % NWG : warp;
  const int gsamp = gw * 512 + lane * 16;
  const int m0 = wk.m0, m1 = m0 + 1;
  const bool has_m1 = m1 < P;
  const uint32_t bar_park = bars + 16 * warp, bar_b = bar_park + 8;
  const uint32_t dst0 = base + warp * WARP_BYTES;                     // this warp's slice of row buffer 0
  if (lane == 0) {
    mbar_init(bar_park, 1);
    mbar_init(bar_b, 1);
    fence_barrier_init();
    prefetch_tensormap(&tmA);
  }
  __syncwarp();
  if (lane == 0) {                                                    // each warp fetches only what it reads itself
    mbar_arrive_expect_tx(bar_park, 2 * WARP_BYTES);
    tma_load_4d(dst0, &tmA, bar_park, 0, 32 * gw, m0, plane0 + j);
    tma_load_4d(dst0 + ROW_BYTES, &tmA, bar_park, 0, 32 * gw, has_m1 ? m1 : m0, plane0 + j);
    mbar_arrive_expect_tx(bar_b, WARP_BYTES);
    tma_load_4d(dst0 + 2 * ROW_BYTES, &tmA, bar_b, 0, 32 * gw, wk.n_begin, plane0 + j);
  }
  // Output recurrence in real arithmetic.  With y = Im(cs w), z = Im(cs zeta w) and zeta^2 = a1 zeta + a2:
  //   V_e = (omf + Im cs) x_e + z_{e-1},  y_e = Im(cs) x_e + z_{e-1},  z_e = Im(cs zeta) x_e + a1 z_{e-1} + a2 y_{e-1}
  // (5 operations per sample instead of 7).  The power-of-two output scale sv rides on the coefficients: exact.
  const float sv = HALF_OUT ? hc::v_scale(*ho.vbound, false) : 1.f;
  const float2 csv = make_float2(cs.x * sv, cs.y * sv);
  const float2 czv = make_float2(csv.x * zeta.x - csv.y * zeta.y, csv.x * zeta.y + csv.y * zeta.x);   // cs zeta sv
  const float a1 = 2.f * zeta.x, a2 = -(zeta.x * zeta.x + zeta.y * zeta.y);
  const float kx = omf * sv + csv.y;
  const float2 pl = zp[lane];                                         // zeta^(16 lane)
  mbar_wait(bar_park, 0, 11);
  int parity = 0;
  for (int n = wk.n_begin; n < wk.n_end; ++n, parity ^= 1) {
    // x0 = Re(A_m0 A_n*), x1 = Re(A_m1 A_n*) on this thread's 16 samples
    float x0[16], x1[16];
    mbar_wait(bar_b, (uint32_t)parity, 12);
#pragma unroll
    for (int c = 0; c < 8; ++c) {                                     // chunk c = samples 2c, 2c + 1
      const int slot = tid * 8 + (c ^ (tid & 7));
      const float4 a0 = rows[slot], a1 = rows[NT * 8 + slot], b = rows[2 * NT * 8 + slot];
      x0[2 * c] = a0.x * b.x + a0.y * b.y;
      x0[2 * c + 1] = a0.z * b.z + a0.w * b.w;
      x1[2 * c] = a1.x * b.x + a1.y * b.y;
      x1[2 * c + 1] = a1.z * b.z + a1.w * b.w;
    }
    __syncwarp();                                                     // the warp is done with the streamed slice
    if (lane == 0 && n + 1 < wk.n_end) {                              // refill it for n + 1 behind the arithmetic
      mbar_arrive_expect_tx(bar_b, WARP_BYTES);
      tma_load_4d(dst0 + 2 * ROW_BYTES, &tmA, bar_b, 0, 32 * gw, n + 1, plane0 + j);
    }
    // chunk total from a zero state: sum_e zeta^(15 - e) x_e
    float2 w0 = make_float2(0.f, 0.f), w1 = w0;
#pragma unroll
    for (int e = 0; e < 16; ++e) {
      w0.x = fmaf(x0[e], zk.re[15 - e], w0.x); w0.y = fmaf(x0[e], zk.im[15 - e], w0.y);
      w1.x = fmaf(x1[e], zk.re[15 - e], w1.x); w1.y = fmaf(x1[e], zk.im[15 - e], w1.y);
    }
    // inclusive scan of the chunk totals inside the warp: T_k = sum_{i<=k} zeta^(16 (k-i)) E_i
#pragma unroll
    for (int d = 1; d < 32; d <<= 1) {
      const float2 pw = zp[d];
      const float r0x = __shfl_up_sync(0xffffffffu, w0.x, d), r0y = __shfl_up_sync(0xffffffffu, w0.y, d);
      const float r1x = __shfl_up_sync(0xffffffffu, w1.x, d), r1y = __shfl_up_sync(0xffffffffu, w1.y, d);
      if (lane >= d) {
        w0 = make_float2(w0.x + pw.x * r0x - pw.y * r0y, w0.y + pw.x * r0y + pw.y * r0x);
        w1 = make_float2(w1.x + pw.x * r1x - pw.y * r1y, w1.y + pw.x * r1y + pw.y * r1x);
      }
    }
    if (lane == 31) { wt[(parity * NW + warp) * 2] = w0; wt[(parity * NW + warp) * 2 + 1] = w1; }
    float2 e0 = make_float2(__shfl_up_sync(0xffffffffu, w0.x, 1), __shfl_up_sync(0xffffffffu, w0.y, 1));
    float2 e1 = make_float2(__shfl_up_sync(0xffffffffu, w1.x, 1), __shfl_up_sync(0xffffffffu, w1.y, 1));
    if (lane == 0) { e0 = make_float2(0.f, 0.f); e1 = e0; }
    __syncthreads();
    if (halo_warp) continue;                                          // its total is published; it writes no output
    {
      const int pw = HALO ? warp - 1 : (warp == 0 ? NW - 1 : warp - 1);   // the warp before this one (periodic)
      const float2 g0 = wt[(parity * NW + pw) * 2], g1 = wt[(parity * NW + pw) * 2 + 1];
      // state before this thread's first sample: exclusive in-warp part + zeta^(16 lane) x the previous warp's total
      w0 = make_float2(e0.x + pl.x * g0.x - pl.y * g0.y, e0.y + pl.x * g0.y + pl.y * g0.x);
      w1 = make_float2(e1.x + pl.x * g1.x - pl.y * g1.y, e1.y + pl.x * g1.y + pl.y * g1.x);
    }
    // second pass from the true state: sv V = sv [(1 - f_R) x + Im(cs w)]
    {
      float y0 = csv.x * w0.y + csv.y * w0.x, z0 = czv.x * w0.y + czv.y * w0.x;
      float y1 = csv.x * w1.y + csv.y * w1.x, z1 = czv.x * w1.y + czv.y * w1.x;
#pragma unroll
      for (int e = 0; e < 16; ++e) {
        const float xa = x0[e], xb = x1[e];
        x0[e] = fmaf(kx, xa, z0);
        x1[e] = fmaf(kx, xb, z1);
        const float ya = fmaf(csv.y, xa, z0), yb = fmaf(csv.y, xb, z1);
        z0 = fmaf(czv.y, xa, fmaf(a1, z0, a2 * y0));
        z1 = fmaf(czv.y, xb, fmaf(a1, z1, a2 * y1));
        y0 = ya; y1 = yb;
      }
    }
    const long long q0 = (long long)m0 * P - (long long)m0 * (m0 - 1) / 2 + (n - m0);
    const long long q1 = (long long)m1 * P - (long long)m1 * (m1 - 1) / 2 + (n - m1);
    const bool st1 = has_m1 && n >= m1;                               // (m1, n) exists only for n >= m1
    if constexpr (HALF_OUT) {
      __half* obase = ho.Vh + j * ho.plane_stride + gsamp;
#pragma unroll
      for (int s = 0; s < 2; ++s) {
        if (s == 1 && !st1) break;
        const float* x = s == 0 ? x0 : x1;
        uint32_t hi[8], lo[8];
#pragma unroll
        for (int k = 0; k < 8; ++k) {
          const float2 v = make_float2(x[2 * k], x[2 * k + 1]);
          const __half2 h = __float22half2_rn(v);
          const float2 f = __half22float2(h);
          const __half2 l = __float22half2_rn(make_float2(v.x - f.x, v.y - f.y));
          hi[k] = *reinterpret_cast<const uint32_t*>(&h);
          lo[k] = *reinterpret_cast<const uint32_t*>(&l);
        }
        __half* row = obase + ho.row(s == 0 ? q0 : q1) * N;
        stg256(row, hi);
        stg256(row + ho.lo_offset, lo);
      }
    } else {
      float* obase = V + j * v_plane_stride + gsamp;
#pragma unroll
      for (int s = 0; s < 2; ++s) {
        if (s == 1 && !st1) break;
        const float* x = s == 0 ? x0 : x1;
        float* row = obase + (s == 0 ? q0 : q1) * N;
        uint32_t u[8];
#pragma unroll
        for (int h = 0; h < 2; ++h) {
#pragma unroll
          for (int k = 0; k < 8; ++k) u[k] = __float_as_uint(x[8 * h + k]);
          stg256(row + 8 * h, u);
        }
      }
    }
  }
}

// ------------------------------------------------------------------------------------------
// a6 (CUDA-core form): U[j][r][t] = sum_q S2[r][q] V[j][q][t], r,q packed pairs (p<=l), (m<=n);
// S2 holds S_plmn with off-diagonal (m<n) columns doubled.
// Plain register-tiled GEMM, C[Q x N] = S2[Q x Q] * V_j[Q x N], one plane per blockIdx.z.
template <typename T, int BM, int BN, int BK, int TM, int TN>
__global__ void __launch_bounds__((BM / TM) * (BN / TN))
k_contract(const T* __restrict__ S2, const T* __restrict__ V, long long v_plane_stride, T* __restrict__ U,
           long long u_plane_stride, int Q, int N) {
  pdl_prologue();
  constexpr int NTH = (BM / TM) * (BN / TN);
  __shared__ T As[BK][BM + 4];
  __shared__ T Bs[BK][BN];
  const T* B = V + blockIdx.z * v_plane_stride;
  T* C = U + blockIdx.z * u_plane_stride;
  const int m0 = blockIdx.y * BM, n0 = blockIdx.x * BN;
  const int tid = threadIdx.x;
  const int tx = tid % (BN / TN), ty = tid / (BN / TN);
  T acc[TM][TN];
#pragma unroll
  for (int i = 0; i < TM; ++i)
#pragma unroll
    for (int jn = 0; jn < TN; ++jn) acc[i][jn] = 0;
  for (int k0 = 0; k0 < Q; k0 += BK) {
    for (int idx = tid; idx < BM * BK; idx += NTH) {
      const int r = idx / BK, kk = idx % BK;
      const int gr = m0 + r, gk = k0 + kk;
      As[kk][r] = (gr < Q && gk < Q) ? S2[(long long)gr * Q + gk] : (T)0;
    }
    for (int idx = tid; idx < BK * BN; idx += NTH) {
      const int kk = idx / BN, c = idx % BN;
      const int gk = k0 + kk, gc = n0 + c;
      Bs[kk][c] = (gk < Q && gc < N) ? B[(long long)gk * N + gc] : (T)0;
    }
    __syncthreads();
#pragma unroll
    for (int kk = 0; kk < BK; ++kk) {
      T a[TM], b[TN];
#pragma unroll
      for (int i = 0; i < TM; ++i) a[i] = As[kk][ty * TM + i];
#pragma unroll
      for (int jn = 0; jn < TN; ++jn) b[jn] = Bs[kk][tx + jn * (BN / TN)];
#pragma unroll
      for (int i = 0; i < TM; ++i)
#pragma unroll
        for (int jn = 0; jn < TN; ++jn) acc[i][jn] += a[i] * b[jn];
    }
    __syncthreads();
  }
#pragma unroll
  for (int i = 0; i < TM; ++i) {
    const int gr = m0 + ty * TM + i;
    if (gr >= Q) continue;
#pragma unroll
    for (int jn = 0; jn < TN; ++jn) {
      const int gc = n0 + tx + jn * (BN / TN);
      if (gc < N) C[(long long)gr * N + gc] = acc[i][jn];
    }
  }
}

// ------------------------------------------------------------------------------------------
// a7: N_p(t) = sum_l U_pl(t) A_l(t), U real symmetric, stored packed: row r(p,l) = p P - p(p-1)/2 + (l-p)
// for p <= l.  grid = (N / TW, n_planes); blockDim = TW * G: thread (tx, g) owns sample t = TW bx + tx
// and modes p = g, g + G, ...; the A tile [P][TW] is staged in shared memory, the accumulator of one
// (p, t) lives in registers, so the U loads of a row are independent and pipeline freely.  Each U value
// is read twice (once as U_pl, once as U_lp) by threads of the same CTA: the second read hits L1/L2.
template <typename T, int TW>
__global__ void __launch_bounds__(512)
k_mode_reduce(const T* __restrict__ U, long long u_plane_stride, const cplx<T>* __restrict__ A,
              long long a_plane_stride, cplx<T>* __restrict__ Nt, long long n_plane_stride, int P, int N) {
  pdl_prologue();
  // TW = samples per CTA (32 / 64 / 128): a narrow tile keeps the CTA's slice of U (Q x TW x 4 B) small enough
  // that its second read (U_lp) still finds the first (U_pl) in L2
  extern __shared__ __align__(16) unsigned char smem_raw[];
  cplx<T>* a_s = reinterpret_cast<cplx<T>*>(smem_raw);        // [P][TW]
  const int tx = threadIdx.x % TW, g = threadIdx.x / TW, G = blockDim.x / TW, j = blockIdx.y;
  const int t0 = blockIdx.x * TW;
  const cplx<T>* Aj = A + j * a_plane_stride + t0;
  for (int i = threadIdx.x; i < P * TW; i += blockDim.x) {
    const int x = i % TW;
    a_s[i] = t0 + x < N ? Aj[(long long)(i / TW) * N + x] : mk((T)0, (T)0);
  }
  __syncthreads();
  const int t = t0 + tx;
  if (t >= N) return;
  const T* Ut = U + j * u_plane_stride + t;
  const cplx<T>* at = a_s + tx;
  for (int p = g; p < P; p += G) {
    T sx = 0, sy = 0;
    long long r = p;                                  // r(0, p)
#pragma unroll 8
    for (int l = 0; l < p; ++l) {                     // column part: U_lp, l < p
      const T u = Ut[r * N];
      const cplx<T> a = at[l * TW];
      sx += u * a.x;
      sy += u * a.y;
      r += P - l - 1;                                 // r(l+1, p) - r(l, p)
    }
#pragma unroll 8
    for (int l = p; l < P; ++l, ++r) {                // row part: U_pl, l >= p; r == r(p, p) here
      const T u = Ut[r * N];
      const cplx<T> a = at[l * TW];
      sx += u * a.x;
      sy += u * a.y;
    }
    Nt[j * n_plane_stride + (long long)p * N + t] = mk(sx, sy);
  }
}

// ------------------------------------------------------------------------------------------
// a7, streaming form (complex64, packed symmetric U): the kernel above reads every U value twice (as U_pl and as
// U_lp), the second time out of L2 if the slice survived there, with 4-byte loads whose latency it cannot hide
// (ncu: 70 % of the stall samples wait on memory, DRAM 38 %).  Here a persistent CTA owns (plane, 16-sample) slices:
// TMA brings the slice's U[Q][16] (64 B per row) and A[P][16] into shared memory behind an mbarrier while the previous
// slice is being reduced (two buffers), so U crosses HBM once and both of its uses are shared-memory reads.
//   thread (t, g): sample t0 + t, modes p = g, g + G, ... (G = blockDim / 16 groups: one mode per thread up to
//   P = 64); accumulators in registers as above.
//   tmU: U [planes][Q][N] fp32, box 16 x rows_box x 1;  tmA: field [planes][P][2 N floats], box 32 floats x P x 1.
//   grid = min(#SM, slices), block = 16 G, dynamic smem = 2 (n_box rows_box 64 + P 128) + 16 (+ alignment).
template <int TW>                                                     // samples per slice: 16 (large Q) or 64
__global__ void __launch_bounds__(1024, 1)
k_mode_reduce_stream(const __grid_constant__ CUtensorMap tmU, const __grid_constant__ CUtensorMap tmA, int plane0_u,
                     int plane0_a, float2* __restrict__ Nt, long long n_plane_stride, int P, int Q, int N,
                     int n_slices, int n_box, int rows_box) {
  using namespace ptx;
  pdl_launch_dependents();
  extern __shared__ unsigned char smem_raw[];
  const uint32_t raw_addr = smem_u32(smem_raw);
  const uint32_t base = (raw_addr + 127u) & ~127u;
  unsigned char* sm = smem_raw + (base - raw_addr);
  // U arrives as n_box boxes of rows_box rows (n_box rows_box >= Q; rows past Q are zero-filled by TMA)
  const uint32_t u_bytes = (uint32_t)(n_box * rows_box) * (4u * TW), a_bytes = (uint32_t)P * (8u * TW),
                 buf_bytes = u_bytes + a_bytes;
  const uint32_t bars = base + 2 * buf_bytes;
  const int tid = threadIdx.x, t = tid % TW, g = tid / TW;
  const int per_plane = N / TW;
  if (tid == 0) {
    mbar_init(bars, 1);
    mbar_init(bars + 8, 1);
    fence_barrier_init();
    prefetch_tensormap(&tmU);
    prefetch_tensormap(&tmA);
  }
  __syncthreads();
  pdl_wait();
  auto issue = [&](int slice, int b) {                               // one thread: fill buffer b with `slice`
    const int pl = slice / per_plane, t0 = (slice - pl * per_plane) * TW;
    const uint32_t dst = base + b * buf_bytes, bar = bars + 8 * b;
    mbar_arrive_expect_tx(bar, buf_bytes);
    for (int k = 0; k < n_box; ++k) tma_load_3d(dst + k * rows_box * (4 * TW), &tmU, bar, t0, rows_box * k, plane0_u + pl);
    tma_load_3d(dst + u_bytes, &tmA, bar, 2 * t0, 0, plane0_a + pl);
  };
  int it = 0;
  if (tid == 0 && (int)blockIdx.x < n_slices) issue(blockIdx.x, 0);
  for (int slice = blockIdx.x; slice < n_slices; slice += gridDim.x, ++it) {
    const int b = it & 1;
    const int next = slice + gridDim.x;
    if (tid == 0 && next < n_slices) issue(next, b ^ 1);             // buffer b ^ 1 was released by the barrier below
    mbar_wait(bars + 8 * b, (uint32_t)((it >> 1) & 1), 21);
    const float* us = reinterpret_cast<const float*>(sm + b * buf_bytes) + t;
    const float2* as = reinterpret_cast<const float2*>(sm + b * buf_bytes + u_bytes) + t;
    const int pl = slice / per_plane, t0 = (slice - pl * per_plane) * TW;
    for (int p = g; p < P; p += (int)blockDim.x / TW) {
      float sx = 0.f, sy = 0.f;
      int r = p;                                                     // r(0, p)
#pragma unroll 4
      for (int l = 0; l < p; ++l) {                                  // column part: U_lp, l < p
        const float u = us[r * TW];
        const float2 a = as[l * TW];
        sx = fmaf(u, a.x, sx);
        sy = fmaf(u, a.y, sy);
        r += P - l - 1;
      }
#pragma unroll 4
      for (int l = p; l < P; ++l, ++r) {                             // row part: U_pl, l >= p; r == r(p, p) here
        const float u = us[r * TW];
        const float2 a = as[l * TW];
        sx = fmaf(u, a.x, sx);
        sy = fmaf(u, a.y, sy);
      }
      Nt[pl * n_plane_stride + (long long)p * N + t0 + t] = make_float2(sx, sy);
    }
    __syncthreads();                                                 // everyone is done with buffer b
  }
}

// ------------------------------------------------------------------------------------------
// a7, general form: N_p(t) = sum_l A_l(t) U_pl(t) with complex, unsymmetric U stored as two blocks of real
// rows: Re U_pl at row p P + l, Im U_pl at row Bp + p P + l.  grid = (N / 128, n_planes), blockDim = 128 G.
template <typename T>
__global__ void __launch_bounds__(512)
k_mode_reduce_gen(const T* __restrict__ U, long long u_plane_stride, const cplx<T>* __restrict__ A,
                  long long a_plane_stride, cplx<T>* __restrict__ Nt, long long n_plane_stride, int P, int Bp, int N) {
  pdl_prologue();
  extern __shared__ __align__(16) unsigned char smem_raw[];
  cplx<T>* a_s = reinterpret_cast<cplx<T>*>(smem_raw);        // [P][128]
  const int tx = threadIdx.x & 127, g = threadIdx.x >> 7, G = blockDim.x >> 7, j = blockIdx.y;
  const int t0 = blockIdx.x * 128;
  const cplx<T>* Aj = A + j * a_plane_stride + t0;
  for (int i = threadIdx.x; i < P * 128; i += blockDim.x) {
    const int x = i & 127;
    a_s[i] = t0 + x < N ? Aj[(long long)(i >> 7) * N + x] : mk((T)0, (T)0);
  }
  __syncthreads();
  const int t = t0 + tx;
  if (t >= N) return;
  const T* Ur = U + j * u_plane_stride + t;
  const T* Ui = Ur + (long long)Bp * N;
  const cplx<T>* at = a_s + tx;
  for (int p = g; p < P; p += G) {
    T sx = 0, sy = 0;
#pragma unroll 4
    for (int l = 0; l < P; ++l) {
      const long long r = (long long)(p * P + l) * N;
      const T ur = Ur[r], ui = Ui[r];
      const cplx<T> a = at[l * 128];
      sx += ur * a.x - ui * a.y;
      sy += ur * a.y + ui * a.x;
    }
    Nt[j * n_plane_stride + (long long)p * N + t] = mk(sx, sy);
  }
}

// ------------------------------------------------------------------------------------------
// a6 + a7 (and a4 when there is no Raman term) for small P in ONE CUDA-core kernel: with Q = P(P+1)/2 < 64 the
// contraction is a 21 x 21 ... 55 x 55 matrix per sample, far below an MMA tile and not GEMM-bound (SURVEY.md
// 8(d) "a6-a7 at P <= 20: plain FP32 ALUs").  Everything here is pointwise in t:
//   U_r(t) = sum_q S2[r][q] V_q(t),  r = (p <= l);   N_p += U_r A_l,  N_l += U_r A_p  (l != p)
// so no U (and with INLINE_PAIRS no V either) ever exists in memory.  SPLIT lanes share a sample: lane s holds the
// streams q = s, s + SPLIT, ... of its sample in registers and takes that share of every inner product, log2 SPLIT
// warp shuffles complete U_r, and every lane keeps N_p (all p) in registers (the triangle is walked with
// compile-time (p, l)).  SPLIT = 1 up to P = 6 (21 streams fit one thread's registers), 4 up to P = 10.  S2 (rows
// padded to a compile-time stride: 128-bit broadcast reads) and the field tile sit in shared memory.
//   grid = (N / TW, planes), block = 128, TW = 128 / SPLIT samples.  PMAX = compile-time bound on P.
//   INLINE_PAIRS: V_q = Re(A_m A_n*) formed here (f_R == 0: a4 is pointwise too), else V is read (a5 ran).
constexpr int kSmallThreads = 128;
template <typename T, int PMAX, int SPLIT, bool INLINE_PAIRS>
__global__ void __launch_bounds__(kSmallThreads)
k_small_contract_reduce(const T* __restrict__ S2, const T* __restrict__ V, long long v_plane_stride,
                        const cplx<T>* __restrict__ A, long long a_plane_stride, cplx<T>* __restrict__ Nt,
                        long long n_plane_stride, const int* __restrict__ pair_m, const int* __restrict__ pair_n,
                        int P, int Q, int N) {
  pdl_prologue();
  constexpr int NTH = kSmallThreads, TW = NTH / SPLIT, QMAX = PMAX * (PMAX + 1) / 2, KQ = (QMAX + SPLIT - 1) / SPLIT,
                QP = (KQ * SPLIT + 3) & ~3;
  extern __shared__ __align__(16) unsigned char smem_raw[];
  T* s2 = reinterpret_cast<T*>(smem_raw);                               // [QMAX][QP], zero-padded
  cplx<T>* a_s = reinterpret_cast<cplx<T>*>(s2 + QMAX * QP);             // [P][TW]
  T* v_s = reinterpret_cast<T*>(a_s + (size_t)P * TW);                   // [Q][TW] (INLINE_PAIRS: unused)
  const int tid = threadIdx.x, j = blockIdx.y, t0 = blockIdx.x * TW;
  for (int i = tid; i < QMAX * QP; i += NTH) {
    const int rr = i / QP, qq = i % QP;
    s2[i] = rr < Q && qq < Q ? S2[rr * Q + qq] : (T)0;
  }
  for (int i = tid; i < P * TW; i += NTH) {
    const int xx = i % TW;
    a_s[i] = t0 + xx < N ? A[j * a_plane_stride + (long long)(i / TW) * N + t0 + xx] : mk((T)0, (T)0);
  }
  const int x = tid / SPLIT, sub = tid % SPLIT;                           // sample, lane among the sample's SPLIT lanes
  T vq[KQ];
  if constexpr (!INLINE_PAIRS) {                                          // this lane's streams straight from V (coalesced over x)
#pragma unroll
    for (int k = 0; k < KQ; ++k) {
      const int q = SPLIT * k + sub;
      vq[k] = q < Q && t0 + x < N ? V[j * v_plane_stride + (long long)q * N + t0 + x] : (T)0;
    }
  }
  __syncthreads();
  if constexpr (INLINE_PAIRS) {
#pragma unroll
    for (int k = 0; k < KQ; ++k) {
      const int q = SPLIT * k + sub;
      vq[k] = (T)0;
      if (q < Q) {
        const cplx<T> am = a_s[pair_m[q] * TW + x], an = a_s[pair_n[q] * TW + x];
        vq[k] = am.x * an.x + am.y * an.y;                                // Re(A_m A_n*)
      }
    }
  }
  T nx[PMAX], ny[PMAX];
#pragma unroll
  for (int p = 0; p < PMAX; ++p) nx[p] = ny[p] = (T)0;
  int r = 0;
#pragma unroll
  for (int p = 0; p < PMAX; ++p) {
    if (p < P) {
      const cplx<T> ap = a_s[p * TW + x];
#pragma unroll
      for (int l = p; l < PMAX; ++l) {
        if (l < P) {
          const T* srow = s2 + r * QP + sub;                              // padded entries are zero: no bound checks
          T up[4] = {(T)0, (T)0, (T)0, (T)0};                            // four independent chains
#pragma unroll
          for (int k = 0; k < KQ; ++k) up[k & 3] += srow[SPLIT * k] * vq[k];
          T u = (up[0] + up[1]) + (up[2] + up[3]);
#pragma unroll
          for (int d = 1; d < SPLIT; d <<= 1) u += __shfl_xor_sync(0xffffffffu, u, d);
          const cplx<T> al = a_s[l * TW + x];
          nx[p] += u * al.x;
          ny[p] += u * al.y;
          if (l != p) {
            nx[l] += u * ap.x;
            ny[l] += u * ap.y;
          }
          ++r;
        }
      }
    }
  }
  if (sub == 0 && t0 + x < N) {
#pragma unroll
    for (int p = 0; p < PMAX; ++p)
      if (p < P) Nt[j * n_plane_stride + (long long)p * N + t0 + x] = mk(nx[p], ny[p]);
  }
}

// ------------------------------------------------------------------------------------------
// a9 + a10: cumulative trapezoid over planes and the per-plane error norms.
//   psi_j^new = psi_0 + dz [G_0/2 + G_1 + .. + G_{j-1} + G_j/2], j = 1..Mc
//   errbuf[2 j] += sum |psi_j^new - psi_j^old|^2,  errbuf[2 j + 1] += sum |psi_j^new|^2
// One thread per (p, w); 256-thread blocks.  Planes are walked eight at a time so that the sixteen loads
// of a batch are in flight together; norms are reduced warp -> shared memory (fp64) -> one global
// atomic per plane per block (a global atomic per warp serialised on 2 Mc addresses: 0.36 ms at config 5).
// Dynamic shared memory: 2 (Mc + 1) doubles.
template <typename T>
__global__ void __launch_bounds__(256)
k_trapz_scan(const cplx<T>* __restrict__ psi0, const cplx<T>* __restrict__ G, cplx<T>* __restrict__ psi,
             long long plane_stride, int Mc, T dz, int first_iter, double* __restrict__ errbuf, long long PN) {
  pdl_prologue();
  extern __shared__ double s_err[];
  for (int i = threadIdx.x; i < 2 * (Mc + 1); i += blockDim.x) s_err[i] = 0.0;
  __syncthreads();
  const long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  const bool live = i < PN;
  const long long ii = live ? i : 0;                 // dead threads read a valid address, write nothing
  const cplx<T> p0 = psi0[ii];
  cplx<T> acc = cscale(G[ii], (T)0.5);
  constexpr int B = 8;
  for (int j0 = 1; j0 <= Mc; j0 += B) {
    cplx<T> g[B], old[B];
#pragma unroll
    for (int b = 0; b < B; ++b) {
      const int j = min(j0 + b, Mc);
      g[b] = G[j * plane_stride + ii];
      old[b] = first_iter ? p0 : psi[j * plane_stride + ii];
    }
#pragma unroll
    for (int b = 0; b < B; ++b) {
      const int j = j0 + b;
      if (j > Mc) break;
      const cplx<T> pn = mk(p0.x + dz * (acc.x + (T)0.5 * g[b].x), p0.y + dz * (acc.y + (T)0.5 * g[b].y));
      acc = cadd(acc, g[b]);
      const cplx<T> d = csub(pn, old[b]);
      T num = live ? d.x * d.x + d.y * d.y : (T)0;
      T den = live ? pn.x * pn.x + pn.y * pn.y : (T)0;
      if (live) psi[j * plane_stride + i] = pn;
#pragma unroll
      for (int o = 16; o > 0; o >>= 1) {
        num += __shfl_xor_sync(0xffffffffu, num, o);
        den += __shfl_xor_sync(0xffffffffu, den, o);
      }
      if ((threadIdx.x & 31) == 0) {
        atomicAdd(&s_err[2 * j], (double)num);
        atomicAdd(&s_err[2 * j + 1], (double)den);
      }
    }
  }
  __syncthreads();
  for (int k = 2 + threadIdx.x; k < 2 * (Mc + 1); k += blockDim.x) atomicAdd(&errbuf[k], s_err[k]);
}

// err = max_j sqrt(num_j / den_j); result -> out[0]; accumulators cleared for the next iteration
// (one warp: lane i takes planes i + 1, i + 33, ...; fmax is exact, so the lane order does not matter)
__device__ __forceinline__ double err_max_over_planes(double* __restrict__ errbuf, int Mc) {
  double e = 0.0;
  for (int j = 1 + (int)threadIdx.x; j <= Mc; j += 32) {
    const double num = errbuf[2 * j], den = errbuf[2 * j + 1];
    e = fmax(e, den > 0.0 ? sqrt(num / den) : 0.0);
    errbuf[2 * j] = 0.0;
    errbuf[2 * j + 1] = 0.0;
  }
#pragma unroll
  for (int d = 16; d > 0; d >>= 1) e = fmax(e, __shfl_xor_sync(0xffffffffu, e, d));
  return e;
}
__global__ void k_err_finalize(double* __restrict__ errbuf, int Mc, double* __restrict__ out) {
  pdl_prologue();
  const double e = err_max_over_planes(errbuf, Mc);
  if (threadIdx.x == 0) out[0] = e;
}

// a10 taken on the device (the loop of PAPER.md:218 as a CUDA-graph WHILE node): the same
// error as k_err_finalize, then the decision the host loop takes after its read-back -- stop when err < tol or
// at the iteration cap -- written to the conditional handle that gates the next pass of the loop body.
// st->it is zeroed by a memset node at the head of every large step; iters / noconv accumulate over a call.
struct LoopStats {
  int it, noconv;
  long long iters;
  double last_err;
  double err_prev, rho_prev;     // stop_rule 1: previous error and previous ratio of this large step
};
// convergence decision shared by the host loop and the device loop: err < tol, or (stop_rule 1, it >= 3) the
// a-posteriori bound err rho / (1 - rho) < tol with rho the larger of the last two error ratios (reading S25)
__host__ __device__ inline bool mpa_converged(double err, double tol, int stop_rule, int it, double err_prev,
                                              double rho_prev, double* rho_out) {
  const double rho_now = err_prev > 0.0 ? err / err_prev : 0.0;
  *rho_out = rho_now;
  if (err < tol) return true;
  if (stop_rule == 1 && it >= 3) {
    const double rho = rho_now > rho_prev ? rho_now : rho_prev;
    if (rho < 1.0 && err * rho / (1.0 - rho) < tol) return true;
  }
  return false;
}
__global__ void k_err_finalize_loop(double* __restrict__ errbuf, int Mc, double* __restrict__ out, double tol, int cap,
                                    int fixed, cudaGraphConditionalHandle handle, LoopStats* __restrict__ st,
                                    int stop_rule) {
  pdl_prologue();
  const double e = err_max_over_planes(errbuf, Mc);
  if (threadIdx.x == 0) {
    out[0] = e;
    const int it = st->it + 1;
    st->it = it;
    st->iters += 1;
    st->last_err = e;
    bool cont;
    if (fixed) {
      cont = it < cap;
    } else {
      const bool first = it == 1;                        // st->it was zeroed at the head of the large step
      double rho = 0.0;
      const bool conv = mpa_converged(e, tol, stop_rule, it, first ? 1e300 : st->err_prev, first ? 1e300 : st->rho_prev,
                                      &rho);
      st->err_prev = e;
      st->rho_prev = first ? 1e300 : rho;
      cont = !conv && it < cap;
      if (!conv && !cont) st->noconv += 1;
    }
    cudaGraphSetConditional(handle, cont ? 1u : 0u);
  }
}

// ------------------------------------------------------------------------------------------
// Plane-axis sharding over several GPUs (the M planes are the parallel axis).
// Shard g owns planes j_lo+1 .. j_hi (shard 0 also plane 0), runs a3-a8 on them and forms its block sum
//   B_g = sum_{j in shard} w_j G_j,  w_0 = 1/2, w_M = 1/2, else 1          (the trapezoid weights of PAPER.md:218)
// One all-gather of the block sums (P N complex each) gives every shard its exclusive prefix sum_{g' < g} B_g',
// from which its planes follow exactly as in k_trapz_scan; sum_g B_g is the whole integral, so every shard can
// advance psi_0 by itself (no broadcast).  The convergence test adds one scalar max all-reduce.
template <typename T>
__global__ void __launch_bounds__(256)
k_shard_block_sum(const cplx<T>* __restrict__ G, long long plane_stride, int j_lo, int j_hi, int Mc,
                  cplx<T>* __restrict__ out, long long PN) {
  pdl_prologue();
  const long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= PN) return;
  cplx<T> acc = j_lo == 0 ? cscale(G[i], (T)0.5) : mk((T)0, (T)0);
  for (int j = j_lo + 1; j <= j_hi; ++j) {
    const cplx<T> g = G[j * plane_stride + i];
    acc = cadd(acc, j == Mc ? cscale(g, (T)0.5) : g);
  }
  out[i] = acc;
}
// start value of shard `shard`'s running sum: G_0 / 2 on the first shard, else the sum of the earlier shards' blocks
template <typename T>
__global__ void __launch_bounds__(256)
k_shard_prefix(const cplx<T>* __restrict__ all_sums, int shard, const cplx<T>* __restrict__ G0,
               cplx<T>* __restrict__ out, long long PN) {
  pdl_prologue();
  const long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= PN) return;
  cplx<T> acc = mk((T)0, (T)0);
  if (shard == 0) acc = cscale(G0[i], (T)0.5);
  for (int g = 0; g < shard; ++g) acc = cadd(acc, all_sums[g * PN + i]);
  out[i] = acc;
}
// a9 + a10 on the shard's planes: psi_j^new = psi_0 + dz [prefix + G_{j_lo+1} + .. + G_{j-1} + G_j / 2]
template <typename T>
__global__ void __launch_bounds__(256)
k_shard_scan(const cplx<T>* __restrict__ psi0, const cplx<T>* __restrict__ G, cplx<T>* __restrict__ psi,
             long long plane_stride, int j_lo, int j_hi, T dz, int first_iter, const cplx<T>* __restrict__ prefix,
             double* __restrict__ errbuf, long long PN) {
  pdl_prologue();
  const long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  const bool live = i < PN;
  const long long ii = live ? i : 0;
  const cplx<T> p0 = psi0[ii];
  cplx<T> acc = prefix[ii];
  for (int j = j_lo + 1; j <= j_hi; ++j) {
    const cplx<T> g = G[j * plane_stride + ii];
    const cplx<T> old = first_iter ? p0 : psi[j * plane_stride + ii];
    const cplx<T> pn = mk(p0.x + dz * (acc.x + (T)0.5 * g.x), p0.y + dz * (acc.y + (T)0.5 * g.y));
    acc = cadd(acc, g);
    const cplx<T> d = csub(pn, old);
    double num = live ? (double)(d.x * d.x + d.y * d.y) : 0.0;
    double den = live ? (double)(pn.x * pn.x + pn.y * pn.y) : 0.0;
    if (live) psi[j * plane_stride + i] = pn;
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
      num += __shfl_xor_sync(0xffffffffu, num, o);
      den += __shfl_xor_sync(0xffffffffu, den, o);
    }
    if ((threadIdx.x & 31) == 0) {
      atomicAdd(&errbuf[2 * j], num);
      atomicAdd(&errbuf[2 * j + 1], den);
    }
  }
}
// a11 from the gathered block sums: psi0_d <- (psi0_d + dz sum_g B_g) exp(D Mc dz), on every shard alike
template <typename T>
__global__ void __launch_bounds__(256)
k_shard_advance(double2* __restrict__ psi0_d, cplx<T>* __restrict__ psi0, const cplx<T>* __restrict__ all_sums,
                int n_shards, double dz, const double2* __restrict__ EM, long long PN, int* __restrict__ step2, int Mc) {
  pdl_prologue();
  const long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (i == 0 && step2) *step2 += 2 * Mc;
  if (i >= PN) return;
  double ax = 0.0, ay = 0.0;
  for (int g = 0; g < n_shards; ++g) {
    const cplx<T> b = all_sums[g * PN + i];
    ax += (double)b.x;
    ay += (double)b.y;
  }
  double2 p = psi0_d[i];
  p.x += dz * ax;
  p.y += dz * ay;
  const double2 e = EM[i];
  const double2 q = make_double2(p.x * e.x - p.y * e.y, p.x * e.y + p.y * e.x);
  psi0_d[i] = q;
  psi0[i] = mk((T)q.x, (T)q.y);
}

// ------------------------------------------------------------------------------------------
// a11: advance the fp64 master state by one large step and refresh its working-precision copy.
//   psi0_d <- (psi0_d + dz [G_0/2 + G_1 + .. + G_{Mc-1} + G_Mc/2]) * exp(D Mc dz)
template <typename T>
__global__ void __launch_bounds__(256)
k_advance(double2* __restrict__ psi0_d, cplx<T>* __restrict__ psi0, const cplx<T>* __restrict__ G,
          long long plane_stride, int Mc, double dz, const double2* __restrict__ EM, long long PN,
          int* __restrict__ step2) {
  pdl_prologue();
  const long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (i == 0 && step2) *step2 += 2 * Mc;               // position along the call, in half small steps (z-profiles)
  if (i >= PN) return;
  double ax = 0.5 * (double)G[i].x, ay = 0.5 * (double)G[i].y;
  for (int j = 1; j < Mc; ++j) {
    const cplx<T> g = G[j * plane_stride + i];
    ax += (double)g.x;
    ay += (double)g.y;
  }
  const cplx<T> gm = G[Mc * plane_stride + i];
  ax += 0.5 * (double)gm.x;
  ay += 0.5 * (double)gm.y;
  double2 p = psi0_d[i];
  p.x += dz * ax;
  p.y += dz * ay;
  const double2 e = EM[i];
  const double2 q = make_double2(p.x * e.x - p.y * e.y, p.x * e.y + p.y * e.x);
  psi0_d[i] = q;
  psi0[i] = mk((T)q.x, (T)q.y);
}

// ------------------------------------------------------------------------------------------
// Serial comparison integrator: the elementwise stages of one RK4IP step in the
// frequency domain.  With E = exp(D h/2), Nh(X) = K F{N[F^-1 X]} (the same a4-a8 kernels, one plane):
//   stage 1: AI = E At;  K1 = h E G;  X = AI + K1/2          (G = Nh(At))
//   stage 2: K2 = h G;  X = AI + K2/2                        (G = Nh(X))
//   stage 3: K3 = h G;  X = E (AI + K3)
//   stage 4: At <- E (AI + K1/6 + K2/3 + K3/3) + h G/6       (fp64 master copy + working copy)
// The interaction-picture form replaces the split-step scheme the paper compares against.
template <typename T>
__global__ void __launch_bounds__(256)
k_rk4_stage(int stage, double2* __restrict__ At_d, cplx<T>* __restrict__ At, const double2* __restrict__ EH,
            const cplx<T>* __restrict__ G, cplx<T>* __restrict__ AI, cplx<T>* __restrict__ K1,
            cplx<T>* __restrict__ K2, cplx<T>* __restrict__ K3, cplx<T>* __restrict__ X, double h, long long PN,
            int* __restrict__ step2) {
  pdl_prologue();
  const long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (i == 0 && stage == 4 && step2) *step2 += 2;
  if (i >= PN) return;
  const double2 e = EH[i];
  const double gx = (double)G[i].x * h, gy = (double)G[i].y * h;
  if (stage == 1) {
    const double2 a = At_d[i];
    const double aix = a.x * e.x - a.y * e.y, aiy = a.x * e.y + a.y * e.x;
    const double k1x = gx * e.x - gy * e.y, k1y = gx * e.y + gy * e.x;
    AI[i] = mk((T)aix, (T)aiy);
    K1[i] = mk((T)k1x, (T)k1y);
    X[i] = mk((T)(aix + 0.5 * k1x), (T)(aiy + 0.5 * k1y));
  } else if (stage == 2) {
    K2[i] = mk((T)gx, (T)gy);
    X[i] = mk((T)((double)AI[i].x + 0.5 * gx), (T)((double)AI[i].y + 0.5 * gy));
  } else if (stage == 3) {
    K3[i] = mk((T)gx, (T)gy);
    const double sx = (double)AI[i].x + gx, sy = (double)AI[i].y + gy;
    X[i] = mk((T)(sx * e.x - sy * e.y), (T)(sx * e.y + sy * e.x));
  } else {
    // AI is recomputed from the fp64 master so that the state never passes through working precision
    const double2 a = At_d[i];
    const double aix = a.x * e.x - a.y * e.y, aiy = a.x * e.y + a.y * e.x;
    const double sx = aix + (double)K1[i].x / 6.0 + ((double)K2[i].x + (double)K3[i].x) / 3.0;
    const double sy = aiy + (double)K1[i].y / 6.0 + ((double)K2[i].y + (double)K3[i].y) / 3.0;
    const double2 r = make_double2(sx * e.x - sy * e.y + gx / 6.0, sx * e.y + sy * e.x + gy / 6.0);
    At_d[i] = r;
    At[i] = mk((T)r.x, (T)r.y);
  }
}

// ------------------------------------------------------------------------------------------
// Terms linear in the field with a frequency-independent P x P matrix (section F; SURVEY.md 8(f)
// NEXT-3): G_j[p] += R-_j[p] sum_n X_j[n][p] (R+_j[n] src_j[n]) per frequency, where R+-_j = exp(+-D_w j dz) =
// E^(+-1) x gain factor rotates between the interaction picture of plane j and the field (tables null: no rotation,
// the RK4IP stages).  X_j = i f(z_j) Q - g_sat W_j: linear coupling C_p = i sum_n Q_np A_n (f: the z-profile of the
// perturbation) and first-order gain saturation (W_j from the plane's time-integrated pair products, k_ext_matrix);
// x_plane_stride = 0 when X is the same for every plane (constant coupling alone).
//   grid = (N / 64, n_planes), block = 256: 64 frequencies x 4 mode groups; the rotated field tile sits in smem.
template <typename T>
__global__ void __launch_bounds__(256)
k_couple(const cplx<T>* __restrict__ src, long long src_plane_stride, const cplx<T>* __restrict__ E,
         const T* __restrict__ gfwd, const T* __restrict__ ginv, const cplx<T>* __restrict__ X,
         long long x_plane_stride, cplx<T>* __restrict__ G, long long plane_stride, int P, int N) {
  pdl_prologue();
  extern __shared__ __align__(16) unsigned char smem_raw[];
  cplx<T>* a_s = reinterpret_cast<cplx<T>*>(smem_raw);        // [P][64]
  const int x = threadIdx.x & 63, g = threadIdx.x >> 6, j = blockIdx.y;
  const int w0 = blockIdx.x * 64, w = w0 + x;
  const cplx<T>* sj = src + j * src_plane_stride;
  const cplx<T>* Ej = E ? E + j * plane_stride : nullptr;
  const cplx<T>* Xj = X + j * x_plane_stride;
  for (int i = threadIdx.x; i < P * 64; i += blockDim.x) {
    const int n = i >> 6, xx = i & 63;
    cplx<T> a = mk((T)0, (T)0);
    if (w0 + xx < N) {
      a = sj[(long long)n * N + w0 + xx];
      if (Ej) a = cmul(a, Ej[(long long)n * N + w0 + xx]);
      if (gfwd) a = cscale(a, gfwd[j * P + n]);
    }
    a_s[i] = a;
  }
  __syncthreads();
  if (w >= N) return;
  for (int p = g; p < P; p += 4) {
    T sx = 0, sy = 0;
    for (int n = 0; n < P; ++n) {
      const cplx<T> q = Xj[n * P + p], a = a_s[n * 64 + x];
      sx += q.x * a.x - q.y * a.y;
      sy += q.x * a.y + q.y * a.x;
    }
    cplx<T> c = mk(sx, sy);
    if (Ej) c = cmulc(c, Ej[(long long)p * N + w]);
    if (ginv) c = cscale(c, ginv[j * P + p]);
    cplx<T>* out = G + j * plane_stride + (long long)p * N + w;
    *out = cadd(*out, c);
  }
}

// Time-integrated pair products of the planes' fields (gain saturation): Ep[j][q] = dt sum_t Re(A_m A_n*),
// q = packed (m <= n).  grid = (Q, n_planes), block = 256; fp64 accumulation.
template <typename T>
__global__ void __launch_bounds__(256)
k_pair_energy(const cplx<T>* __restrict__ A, long long a_plane_stride, const int* __restrict__ pair_m,
              const int* __restrict__ pair_n, T* __restrict__ Ep, int Q, int N, double dt) {
  pdl_prologue();
  __shared__ double red[8];
  const int q = blockIdx.x, j = blockIdx.y;
  const cplx<T>* am = A + j * a_plane_stride + (long long)pair_m[q] * N;
  const cplx<T>* an = A + j * a_plane_stride + (long long)pair_n[q] * N;
  double s = 0.0;
  for (int t = threadIdx.x; t < N; t += 256) {
    const cplx<T> a = am[t], b = an[t];
    s += (double)(a.x * b.x + a.y * b.y);
  }
#pragma unroll
  for (int d = 16; d > 0; d >>= 1) s += __shfl_xor_sync(0xffffffffu, s, d);
  if ((threadIdx.x & 31) == 0) red[threadIdx.x >> 5] = s;
  __syncthreads();
  if (threadIdx.x == 0) {
    double tot = 0.0;
    for (int k = 0; k < 8; ++k) tot += red[k];
    Ep[(long long)j * Q + q] = (T)(tot * dt);
  }
}

// Per-plane matrix of the linear extra terms: X_j[n][p] = i f(z_j) Q_np - g_sat W_j,np with
// W_j,pl = sum_mn S_plmn E_j,mn = sum_q S2[r(p,l)][q] Ep[j][q] (real, symmetric; S2 carries the m < n doubling).
// f(z_j) = fprof[*step2 + 2 (j0 + j) + f_off] (profile sampled every dz / 2 from the start of the call; *step2 = twice the
// small steps already taken, kept on the device by k_advance / k_rk4_stage), 1 without a profile.
//   grid = n_planes, block = 256.  Qc, Ep, fprof may be null (term absent).
template <typename T>
__global__ void __launch_bounds__(256)
k_ext_matrix(const cplx<T>* __restrict__ Qc, const T* __restrict__ S2, const T* __restrict__ Ep, T g_sat,
             const double* __restrict__ fprof, int n_fprof, const int* __restrict__ step2, int j0, int f_off,
             cplx<T>* __restrict__ X, int P, int Q) {
  pdl_prologue();
  const int j = blockIdx.x;
  T f = (T)1;
  if (fprof) {
    int idx = (step2 ? *step2 : 0) + 2 * (j0 + j) + f_off;
    idx = idx < 0 ? 0 : (idx >= n_fprof ? n_fprof - 1 : idx);
    f = (T)fprof[idx];
  }
  for (int i = threadIdx.x; i < P * P; i += 256) {
    const int n = i / P, p = i - n * P;
    cplx<T> x = mk((T)0, (T)0);
    if (Qc) x = mk(-f * Qc[i].y, f * Qc[i].x);                    // i f Q_np
    if (Ep) {
      const int a = n < p ? n : p, b = n < p ? p : n;
      const long long r = (long long)a * P - (long long)a * (a - 1) / 2 + (b - a);
      const T* srow = S2 + r * Q;
      const T* e = Ep + (long long)j * Q;
      T w = (T)0;
      for (int q = 0; q < Q; ++q) w += srow[q] * e[q];
      x.x -= g_sat * w;
    }
    X[(long long)j * P * P + i] = x;
  }
}

// ------------------------------------------------------------------------------------------
// Eq. 2 on the GPU: S_plmn is the Gram matrix of the pair functions
// Phi_r = F_p F_l, r = (p <= l), on the quadrature grid: Gram[r][q] = sum_g Phi_r(g) Phi_q(g).  The product runs on
// the same kind::f16 tcgen05 kernel as a6 (K = grid points); these two kernels prepare its operands from the fp64
// mode fields F[P][G].
//   k_pair_fields_t: A operand, PhiT[g][Npad] fp32 (pair index contiguous, zero beyond Q) -> k_v_encode splits it.
//   k_pair_fields_b: B operand, rows r of Phi as fp16 hi / lo [Rp][G] scaled per row by 2^(14 - e_r) (exact), with
//                    rscale[r] = 2^-(14 - e_r); one CTA per row (row maximum first, then the split).
__global__ void __launch_bounds__(256)
k_pair_fields_t(const double* __restrict__ F, long long G, const int* __restrict__ pair_p, const int* __restrict__ pair_l,
                int Q, int Npad, float* __restrict__ PhiT) {
  pdl_prologue();
  const long long total = G * Npad;
  for (long long i = (long long)blockIdx.x * 256 + threadIdx.x; i < total; i += (long long)gridDim.x * 256) {
    const long long g = i / Npad;
    const int r = (int)(i - g * Npad);
    PhiT[i] = r < Q ? (float)(F[pair_p[r] * G + g] * F[pair_l[r] * G + g]) : 0.f;
  }
}
__global__ void __launch_bounds__(256)
k_pair_fields_b(const double* __restrict__ F, long long G, const int* __restrict__ pair_p, const int* __restrict__ pair_l,
                int Q, __half* __restrict__ hi, __half* __restrict__ lo, float* __restrict__ rscale) {
  pdl_prologue();
  __shared__ double red[8];
  __shared__ int s_sh;
  const int r = blockIdx.x;
  __half* hrow = hi + (long long)r * G;
  __half* lrow = lo + (long long)r * G;
  if (r >= Q) {                                                        // padded rows of the r-tiles: zero
    for (long long g = threadIdx.x; g < G; g += 256) { hrow[g] = __float2half_rn(0.f); lrow[g] = __float2half_rn(0.f); }
    if (threadIdx.x == 0) rscale[r] = 1.f;
    return;
  }
  const double* fp = F + pair_p[r] * G;
  const double* fl = F + pair_l[r] * G;
  double m = 0.0;
  for (long long g = threadIdx.x; g < G; g += 256) m = fmax(m, fabs(fp[g] * fl[g]));
#pragma unroll
  for (int d = 16; d > 0; d >>= 1) m = fmax(m, __shfl_xor_sync(0xffffffffu, m, d));
  if ((threadIdx.x & 31) == 0) red[threadIdx.x >> 5] = m;
  __syncthreads();
  if (threadIdx.x == 0) {
    double amax = 0.0;
    for (int k = 0; k < 8; ++k) amax = fmax(amax, red[k]);
    int e = 0;
    if (amax > 0.0) frexp(amax, &e);
    int sh = amax > 0.0 ? hc::V_RANGE_LOG2 - e : 0;
    sh = sh > 120 ? 120 : (sh < -120 ? -120 : sh);
    s_sh = sh;
    rscale[r] = (float)ldexp(1.0, -sh);
  }
  __syncthreads();
  const int sh = s_sh;
  for (long long g = threadIdx.x; g < G; g += 256) {
    const double v = ldexp(fp[g] * fl[g], sh);
    const __half h = __float2half_rn((float)v);
    hrow[g] = h;
    lrow[g] = __float2half_rn((float)(v - (double)__half2float(h)));
  }
}

// Device-side ends of the Eq. 2 pipeline for gmmnlse_overlap_tensor_noalloc (no host round trip):
//   k_normalise_modes: Fn[p][g] = F[p][g] / sqrt(sum_g F[p][g]^2 dA), one CTA per mode; CTA 0 also writes the packed
//                      pair index arrays (p <= l).  A mode of zero norm gives non-finite output (no host check here).
//   k_expand_gram:     S[p][l][m][n] = dA (Gram[r(p,l)][q(m,n)] + Gram[q][r]) / 2 from the [Q][ld] Gram matrix.
__global__ void __launch_bounds__(256)
k_normalise_modes(const double* __restrict__ F, long long G, double dA, int P, double* __restrict__ Fn,
                  int* __restrict__ pair_p, int* __restrict__ pair_l) {
  pdl_prologue();
  __shared__ double red[8];
  __shared__ double s_inv;
  const int p = blockIdx.x;
  const double* f = F + p * G;
  double acc = 0.0;
  for (long long g = threadIdx.x; g < G; g += 256) acc += f[g] * f[g];
#pragma unroll
  for (int d = 16; d > 0; d >>= 1) acc += __shfl_xor_sync(0xffffffffu, acc, d);
  if ((threadIdx.x & 31) == 0) red[threadIdx.x >> 5] = acc;
  __syncthreads();
  if (threadIdx.x == 0) {
    double tot = 0.0;
    for (int k = 0; k < 8; ++k) tot += red[k];
    s_inv = 1.0 / sqrt(tot * dA);
  }
  __syncthreads();
  const double inv = s_inv;
  for (long long g = threadIdx.x; g < G; g += 256) Fn[p * G + g] = f[g] * inv;
  if (p == 0 && threadIdx.x == 0) {
    int q = 0;
    for (int a = 0; a < P; ++a)
      for (int b = a; b < P; ++b, ++q) { pair_p[q] = a; pair_l[q] = b; }
  }
}
__global__ void __launch_bounds__(256)
k_expand_gram(const float* __restrict__ gram, int ld, int P, double dA, double* __restrict__ S) {
  pdl_prologue();
  const int P2 = P * P, total = P2 * P2;
  for (int i = blockIdx.x * 256 + threadIdx.x; i < total; i += gridDim.x * 256) {
    const int pl = i / P2, mn = i - pl * P2;
    const int p = pl / P, l = pl - p * P, m = mn / P, n = mn - m * P;
    const int a = p < l ? p : l, b = p < l ? l : p, c = m < n ? m : n, d = m < n ? n : m;
    const int r = a * P - a * (a - 1) / 2 + (b - a), q = c * P - c * (c - 1) / 2 + (d - c);
    S[i] = 0.5 * ((double)gram[r * ld + q] + (double)gram[q * ld + r]) * dA;
  }
}

template <typename TI, typename TO>
__global__ void __launch_bounds__(256) k_convert(const TI* __restrict__ in, TO* __restrict__ out, long long n) {
  pdl_prologue();
  const long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (i < n) out[i] = (TO)in[i];
}

}  // namespace gm
