// One-CTA power-of-two FFT: Stockham autosort passes, 16 elements per thread held in
// registers, one padded shared-memory exchange between passes.
//
// Convention (reading S1): DIR = +1 is "to frequency",  X_k = sum_n x_n exp(+2 pi i k n/N);
// DIR = -1 is "to time", exp(-2 pi i k n/N).  Both un-normalised; callers fold 1/N into a table.
//
// Pass structure (restated from the standard Stockham formulation): with Ns = product of the
// radices already applied, butterfly j (0 <= j < N/R) reads x[j + r N/R], r = 0..R-1, multiplies
// by w^(r (j mod Ns)), w = exp(DIR 2 pi i/(Ns R)), takes an in-order R-point DFT and writes
// y[(j / Ns) Ns R + (j mod Ns) + r Ns].  With N/16 threads, thread `tid` owns butterflies
// j = tid + i N/16 and therefore always reads the 16 elements x[tid + e N/16]: reads are
// conflict-free; writes are made conflict-free by the pad  phys(a) = a + (a >> 4).
// First pass: radix 2^(log2N mod 4) (no twiddles, Ns = 1), then radix-16 passes.
#pragma once
#include "cx.cuh"

namespace gm {

constexpr double kCos16[16] = {1.0, 0.92387953251128673848, 0.70710678118654752440, 0.38268343236508977173,
                               0.0, -0.38268343236508977173, -0.70710678118654752440, -0.92387953251128673848,
                               -1.0, -0.92387953251128673848, -0.70710678118654752440, -0.38268343236508977173,
                               0.0, 0.38268343236508977173, 0.70710678118654752440, 0.92387953251128673848};
constexpr double kSin16[16] = {0.0, 0.38268343236508977173, 0.70710678118654752440, 0.92387953251128673848,
                               1.0, 0.92387953251128673848, 0.70710678118654752440, 0.38268343236508977173,
                               0.0, -0.38268343236508977173, -0.70710678118654752440, -0.92387953251128673848,
                               -1.0, -0.92387953251128673848, -0.70710678118654752440, -0.38268343236508977173};

// a *= exp(DIR 2 pi i M / 16), M a compile-time constant
template <typename T, int DIR, int M>
__device__ __forceinline__ cplx<T> mul_w16(cplx<T> a) {
  constexpr int m = M & 15;
  if constexpr (m == 0) return a;
  else if constexpr (m == 4) return cmul_i<DIR>(a);
  else if constexpr (m == 8) return mk(-a.x, -a.y);
  else if constexpr (m == 12) return cmul_i<-DIR>(a);
  else {
    constexpr T c = (T)kCos16[m];
    constexpr T s = (T)(DIR > 0 ? kSin16[m] : -kSin16[m]);
    return mk(a.x * c - a.y * s, a.x * s + a.y * c);
  }
}

template <typename T, int DIR>
__device__ __forceinline__ void dft2(cplx<T>& a0, cplx<T>& a1) {
  cplx<T> t = a0;
  a0 = cadd(t, a1);
  a1 = csub(t, a1);
}

// in-order 4-point DFT, W4 = exp(DIR i pi/2)
template <typename T, int DIR>
__device__ __forceinline__ void dft4(cplx<T>& a0, cplx<T>& a1, cplx<T>& a2, cplx<T>& a3) {
  cplx<T> t0 = cadd(a0, a2), t1 = csub(a0, a2), t2 = cadd(a1, a3), t3 = cmul_i<DIR>(csub(a1, a3));
  a0 = cadd(t0, t2);
  a2 = csub(t0, t2);
  a1 = cadd(t1, t3);
  a3 = csub(t1, t3);
}

template <typename T, int R, int DIR> struct Dft;
template <typename T, int DIR> struct Dft<T, 2, DIR> {
  static __device__ __forceinline__ void run(cplx<T>* a) { dft2<T, DIR>(a[0], a[1]); }
};
template <typename T, int DIR> struct Dft<T, 4, DIR> {
  static __device__ __forceinline__ void run(cplx<T>* a) { dft4<T, DIR>(a[0], a[1], a[2], a[3]); }
};
// 8 = 4 x 2:  n = 2 n1 + n2,  k = k1 + 4 k2
template <typename T, int DIR> struct Dft<T, 8, DIR> {
  static __device__ __forceinline__ void run(cplx<T>* a) {
    dft4<T, DIR>(a[0], a[2], a[4], a[6]);          // n2 = 0 -> b0[k1] in a[0],a[2],a[4],a[6]
    dft4<T, DIR>(a[1], a[3], a[5], a[7]);          // n2 = 1 -> b1[k1]
    cplx<T> b1 = mul_w16<T, DIR, 2>(a[3]), b2 = mul_w16<T, DIR, 4>(a[5]), b3 = mul_w16<T, DIR, 6>(a[7]);
    cplx<T> x0 = cadd(a[0], a[1]), x4 = csub(a[0], a[1]);
    cplx<T> x1 = cadd(a[2], b1), x5 = csub(a[2], b1);
    cplx<T> x2 = cadd(a[4], b2), x6 = csub(a[4], b2);
    cplx<T> x3 = cadd(a[6], b3), x7 = csub(a[6], b3);
    a[0] = x0; a[1] = x1; a[2] = x2; a[3] = x3; a[4] = x4; a[5] = x5; a[6] = x6; a[7] = x7;
  }
};
// 16 = 4 x 4:  n = 4 n1 + n2,  k = k1 + 4 k2
template <typename T, int DIR> struct Dft<T, 16, DIR> {
  static __device__ __forceinline__ void run(cplx<T>* a) {
    dft4<T, DIR>(a[0], a[4], a[8], a[12]);         // n2 = 0: b[0][k1] at a[4 k1]
    dft4<T, DIR>(a[1], a[5], a[9], a[13]);         // n2 = 1: b[1][k1] at a[4 k1 + 1]
    dft4<T, DIR>(a[2], a[6], a[10], a[14]);
    dft4<T, DIR>(a[3], a[7], a[11], a[15]);
    // twiddle b[n2][k1] *= W16^(n2 k1)
    a[5] = mul_w16<T, DIR, 1>(a[5]);  a[6] = mul_w16<T, DIR, 2>(a[6]);   a[7] = mul_w16<T, DIR, 3>(a[7]);
    a[9] = mul_w16<T, DIR, 2>(a[9]);  a[10] = mul_w16<T, DIR, 4>(a[10]); a[11] = mul_w16<T, DIR, 6>(a[11]);
    a[13] = mul_w16<T, DIR, 3>(a[13]); a[14] = mul_w16<T, DIR, 6>(a[14]); a[15] = mul_w16<T, DIR, 9>(a[15]);
    // outer DFT over n2 for each k1: inputs a[4 k1 + n2] -> X[k1 + 4 k2]
    dft4<T, DIR>(a[0], a[1], a[2], a[3]);          // k1 = 0 -> X[0],X[4],X[8],X[12]
    dft4<T, DIR>(a[4], a[5], a[6], a[7]);          // k1 = 1 -> X[1],X[5],X[9],X[13]
    dft4<T, DIR>(a[8], a[9], a[10], a[11]);
    dft4<T, DIR>(a[12], a[13], a[14], a[15]);
    // now a[4 k1 + k2] = X[k1 + 4 k2]: transpose the 4x4 index to get in-order output
    cplx<T> t;
    t = a[1]; a[1] = a[4]; a[4] = t;   t = a[2]; a[2] = a[8]; a[8] = t;   t = a[3]; a[3] = a[12]; a[12] = t;
    t = a[6]; a[6] = a[9]; a[9] = t;   t = a[7]; a[7] = a[13]; a[13] = t; t = a[11]; a[11] = a[14]; a[14] = t;
  }
};

// DFT16 of a[r] w^r (the twiddled butterfly of a radix-16 Stockham pass), given w1 = w and w4 = w^4.
// With r = 4 r1 + r2, k = k1 + 4 k2:
//   X[k1 + 4 k2] = sum_r2 W4^(r2 k2) [ w^r2 W16^(r2 k1) sum_r1 W4^(r1 k1) (w^4)^r1 a[4 r1 + r2] ],
// so only six twiddle values are ever needed (w^4, w^8, w^12, then w, w^2, w^3), three at a time: the
// register peak stays ~20 below the form that first builds w^1..w^15.
template <typename T, int DIR>
__device__ __forceinline__ void dft16_twiddled(cplx<T>* a, cplx<T> w1, cplx<T> w4) {
  {
    const cplx<T> w8 = cmul(w4, w4);
#pragma unroll
    for (int r2 = 0; r2 < 4; ++r2) {
      a[4 + r2] = cmul(a[4 + r2], w4);
      a[8 + r2] = cmul(a[8 + r2], w8);
    }
    const cplx<T> w12 = cmul(w8, w4);
#pragma unroll
    for (int r2 = 0; r2 < 4; ++r2) a[12 + r2] = cmul(a[12 + r2], w12);
  }
  dft4<T, DIR>(a[0], a[4], a[8], a[12]);           // r2 = 0: b[0][k1] at a[4 k1]
  dft4<T, DIR>(a[1], a[5], a[9], a[13]);
  dft4<T, DIR>(a[2], a[6], a[10], a[14]);
  dft4<T, DIR>(a[3], a[7], a[11], a[15]);
  {
    const cplx<T> w2 = cmul(w1, w1);
#pragma unroll
    for (int k1 = 0; k1 < 4; ++k1) {
      a[4 * k1 + 1] = cmul(a[4 * k1 + 1], w1);
      a[4 * k1 + 2] = cmul(a[4 * k1 + 2], w2);
    }
    const cplx<T> w3 = cmul(w2, w1);
#pragma unroll
    for (int k1 = 0; k1 < 4; ++k1) a[4 * k1 + 3] = cmul(a[4 * k1 + 3], w3);
  }
  a[5] = mul_w16<T, DIR, 1>(a[5]);  a[6] = mul_w16<T, DIR, 2>(a[6]);   a[7] = mul_w16<T, DIR, 3>(a[7]);
  a[9] = mul_w16<T, DIR, 2>(a[9]);  a[10] = mul_w16<T, DIR, 4>(a[10]); a[11] = mul_w16<T, DIR, 6>(a[11]);
  a[13] = mul_w16<T, DIR, 3>(a[13]); a[14] = mul_w16<T, DIR, 6>(a[14]); a[15] = mul_w16<T, DIR, 9>(a[15]);
  dft4<T, DIR>(a[0], a[1], a[2], a[3]);            // k1 = 0 -> X[0],X[4],X[8],X[12]
  dft4<T, DIR>(a[4], a[5], a[6], a[7]);
  dft4<T, DIR>(a[8], a[9], a[10], a[11]);
  dft4<T, DIR>(a[12], a[13], a[14], a[15]);
  cplx<T> t;                                       // a[4 k1 + k2] = X[k1 + 4 k2] -> natural order
  t = a[1]; a[1] = a[4]; a[4] = t;   t = a[2]; a[2] = a[8]; a[8] = t;   t = a[3]; a[3] = a[12]; a[12] = t;
  t = a[6]; a[6] = a[9]; a[9] = t;   t = a[7]; a[7] = a[13]; a[13] = t; t = a[11]; a[11] = a[14]; a[14] = t;
}

__host__ __device__ constexpr int fft_hibit(int r) { int b = 1; while (b * 2 <= r) b *= 2; return b; }
__device__ __forceinline__ int fft_pad(int a) { return a + (a >> 4); }
__host__ __device__ constexpr int fft_smem_elems(int N) { return N + (N >> 4); }

// twiddles + butterflies of one pass, in registers.  v[e] = x[tid + e N/16] on entry; on exit the
// r-th output of butterfly i sits in v[i + r (16/R)].
template <typename T, int LOG2N, int DIR, int LOGR, int LOGNS>
__device__ __forceinline__ void fft_pass(cplx<T> (&v)[16], const cplx<T>* __restrict__ tw, int tid) {
  constexpr int R = 1 << LOGR, NB = 16 / R, NT = (1 << LOG2N) / 16, NS = 1 << LOGNS;
#pragma unroll
  for (int i = 0; i < NB; ++i) {
    cplx<T> a[R];
#pragma unroll
    for (int r = 0; r < R; ++r) a[r] = v[i + r * NB];
    if constexpr (LOGNS > 0 && LOGR == 4) {
      const int k = (tid + i * NT) & (NS - 1);
      constexpr int SH = LOG2N - LOGNS - LOGR;     // table index of w^1 is k << SH
      cplx<T> w1 = tw[k << SH], w4 = tw[(4 * k) << SH];
      if (DIR < 0) { w1.y = -w1.y; w4.y = -w4.y; }
      dft16_twiddled<T, DIR>(a, w1, w4);
#pragma unroll
      for (int r = 0; r < R; ++r) v[i + r * NB] = a[r];
      continue;
    } else if constexpr (LOGNS > 0) {
      const int k = (tid + i * NT) & (NS - 1);
      constexpr int SH = LOG2N - LOGNS - LOGR;     // table index of w^1 is k << SH
      cplx<T> w[R];
      // looked-up powers 1,2,4,8; the others are products of at most three looked-up values
#pragma unroll
      for (int b = 1; b < R; b <<= 1) {
        w[b] = tw[(k * b) << SH];
        if (DIR < 0) w[b].y = -w[b].y;
      }
#pragma unroll
      for (int r = 3; r < R; ++r) {
        const int hb = fft_hibit(r);                   // compile-time after unrolling
        if (r != hb) w[r] = cmul(w[hb], w[r - hb]);
      }
#pragma unroll
      for (int r = 1; r < R; ++r) a[r] = cmul(a[r], w[r]);
    }
    Dft<T, R, DIR>::run(a);
#pragma unroll
    for (int r = 0; r < R; ++r) v[i + r * NB] = a[r];
  }
}

// destination (natural index within this pass's output) of output r of butterfly i
template <int LOG2N, int LOGR, int LOGNS>
__device__ __forceinline__ int fft_dst(int tid, int i, int r) {
  constexpr int NT = (1 << LOG2N) / 16, NS = 1 << LOGNS;
  const int j = tid + i * NT;
  return (((j >> LOGNS) << (LOGNS + LOGR)) | (j & (NS - 1))) + (r << LOGNS);
}

template <typename T, int LOG2N, int DIR, int LOGR, int LOGNS, typename StoreF>
__device__ __forceinline__ void fft_tail(cplx<T> (&v)[16], cplx<T>* sm, const cplx<T>* __restrict__ tw,
                                         int tid, StoreF& store) {
  constexpr int R = 1 << LOGR, NB = 16 / R, NT = (1 << LOG2N) / 16;
  fft_pass<T, LOG2N, DIR, LOGR, LOGNS>(v, tw, tid);
  if constexpr (LOGNS + LOGR == LOG2N) {            // last pass: hand the results to the caller
#pragma unroll
    for (int i = 0; i < NB; ++i)
#pragma unroll
      for (int r = 0; r < R; ++r) store(fft_dst<LOG2N, LOGR, LOGNS>(tid, i, r), v[i + r * NB]);
  } else {
#pragma unroll
    for (int i = 0; i < NB; ++i)
#pragma unroll
      for (int r = 0; r < R; ++r) sm[fft_pad(fft_dst<LOG2N, LOGR, LOGNS>(tid, i, r))] = v[i + r * NB];
    __syncthreads();
#pragma unroll
    for (int e = 0; e < 16; ++e) v[e] = sm[fft_pad(tid + e * NT)];
    __syncthreads();
    fft_tail<T, LOG2N, DIR, 4, LOGNS + LOGR, StoreF>(v, sm, tw, tid, store);
  }
}

// Whole transform of one row by one CTA of N/16 threads.
//   load(n)      -> input element n (natural order); called for n = tid + e N/16
//   store(k, X)  <- output element k (natural order)
// `sm` holds fft_smem_elems(N) elements and may be the memory `load` reads / `store` writes,
// provided the caller synchronises before the call when `load` reads data other threads wrote.
template <typename T, int LOG2N, int DIR, typename LoadF, typename StoreF>
__device__ __forceinline__ void block_fft(cplx<T>* sm, const cplx<T>* __restrict__ tw, LoadF load, StoreF store) {
  static_assert(LOG2N >= 4, "N >= 16");
  constexpr int NT = (1 << LOG2N) / 16, REM = LOG2N & 3;
  const int tid = threadIdx.x;
  cplx<T> v[16];
#pragma unroll
  for (int e = 0; e < 16; ++e) v[e] = load(tid + e * NT);
  if constexpr (LOG2N == 4) {
    // single thread, single radix-16 pass
    fft_tail<T, LOG2N, DIR, 4, 0, StoreF>(v, sm, tw, tid, store);
  } else {
    __syncthreads();     // `load` may have read `sm`; the first pass writes it
    if constexpr (REM != 0) fft_tail<T, LOG2N, DIR, REM, 0, StoreF>(v, sm, tw, tid, store);
    else fft_tail<T, LOG2N, DIR, 4, 0, StoreF>(v, sm, tw, tid, store);
  }
}

}  // namespace gm
