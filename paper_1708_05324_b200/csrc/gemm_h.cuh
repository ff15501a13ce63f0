// a6 on the tensor cores with fp16 split operands: U[j][r][t] = sum_q S2[r][q] V[j][q][t]  (the
// sum over m,n of Eq. 1) as a kind::f16 tcgen05 GEMM, twice the MMA rate of the 3xTF32 form of
// gemm_tc.cuh at the same 22 mantissa bits.
//
// An fp16 has the mantissa of a TF32 (10 bits + hidden one) but only 5 exponent bits, so both operands are
// scaled by powers of two (exact) into its range before they are split:
//   V' = sV V,  sV = 2^(14 - e) with bound < 2^e, `bound` a device-side upper bound on |V| over the launch
//        (written before the pair kernel runs: max |A|^2 times the plan's stream gain);
//   V' = Vh + Vl,  Vh = fp16(V'), Vl = fp16(V' - Vh)  -- written by the pair kernels straight into HBM as two
//        fp16 arrays (the same bytes as one fp32 array), so this kernel has no converter warps and TMA feeds
//        the MMA directly;
//   S2[r][:] sS[r] = Sh + Sl likewise on the host from fp64, sS[r] = 2^(14 - e_r) per output row.
// Values below 2^-14 of the scaled range go subnormal (the tensor core honours fp16 subnormals: measured),
// i.e. the absolute resolution is 2^-24 on a range of 2^14: 2^-38 of the largest |V|, far below the
// 2^-22 relative error of the split itself.
//   D += Vh Sl + Vl Sh + Vh Sh;   U = D / (sV sS[r])   (the scales are undone in the epilogue, exactly).
// Two-level accumulation as in gemm_tc.cuh (kind::f16 truncates its fp32 accumulate the same way: measured
// -5.5e-6 mean at K = 1024): a TMEM accumulator holds `kchunk` k-blocks, the epilogue warps add the chunks in
// registers.  The default chunk is 4 k-blocks = 128 q = 24 tensor-core accumulates, the count the TF32 form
// has in its 64 q (K = 8 per MMA there, 16 here); draining 128 lanes x 208 columns costs about as much
// tensor-memory read time as 64 q of MMAs, so shorter chunks make the drain the pace (measured at config 5:
// 0.94 ms per launch with 64-q chunks, 0.82 with 128, 0.72 with no chunking).
//
// Orientation as gemm_tc.cuh: M = t (128 per CTA), N = r (NT <= 208), K = q in blocks of BK = 32.
//   A = V^T is MN-major (t contiguous): rows of 64 t (128 B, SWIZZLE_128B) per q, 8-q groups 1024 B apart
//   (SBO), 64-t groups one TMA box (BK * 128 B) apart (LBO)  -- measured exact on B200 for kind::f16.
//   B = S2 is K-major: rows of 32 q (64 B, SWIZZLE_64B), 8-row groups 512 B apart.
// Warp roles (448 threads): warp 0 TMA producer, warp 1 MMA issuer + TMEM allocator, warps 2-13 epilogue
// (three per TMEM lane group).
#pragma once
#include <cuda.h>
#include <cuda_fp16.h>

#include "cx.cuh"
#include "ptx_sm100.cuh"

namespace gm {
namespace hc {

constexpr int BK = 32;                                  // q per k-block
constexpr int TM = 128;                                 // t per CTA
constexpr int NUM_EPI_WARPS = 12;
constexpr int NTHREADS = 32 * (2 + NUM_EPI_WARPS);      // 448
constexpr int EPI_COLS = 72;                            // columns per epilogue warp (default): NT <= 208
constexpr int EPI_COLS_WIDE = 80;                       // wide instantiation: NT <= 240, one r-tile for Q <= 240
constexpr int EPI_ROUND = 2;                            // tcgen05.ld groups (8 columns each) in flight per wait
constexpr int A_BYTES = TM * BK * 2;                    // 8 KiB: one A tile (hi or lo)
constexpr int MAX_STAGES = 8;
constexpr int TMEM_COLS = 512;
constexpr int ACC_COLS = 256;
constexpr int V_RANGE_LOG2 = 14;                        // scaled operands stay below 2^14 (fp16 max 65504)

// sV and 1/sV from the bound on |V| (both exact powers of two); bound == 0 or not finite -> 1
__host__ __device__ inline float v_scale(float bound, bool inverse) {
  if (!(bound > 0.f) || !(bound < 3.0e38f)) return 1.f;
  int e;
  frexpf(bound, &e);                                    // bound = m 2^e, 0.5 <= m < 1
  e = V_RANGE_LOG2 - e;
  e = e > 100 ? 100 : (e < -100 ? -100 : e);
  return ldexpf(1.f, inverse ? -e : e);
}

struct Params {
  float* U;                    // [plane][Q][N] fp32 (OUT_H == false)
  __half* Zh;                  // OUT_H: [plane][2][Q][N] halves (hi rows then lo rows), scaled by sZ = v_scale(zgain * bound)
  long long u_plane_stride;    // elements of the output type (OUT_H: halves)
  const float* rscale;         // [n_rt * NT] 1 / sS[r]
  const float* vbound;         // device scalar: bound on |V| of this launch
  float bound_gain;            // the A operand was scaled by v_scale(bound_gain * *vbound)
  float zgain;                 // OUT_H: |Z| <= zgain * *vbound
  int Q, N, NT, KB, n_rt, t_tiles, total_tiles, plane0, stages, kchunk;
  // block-sparse form (options.contraction = 9; all three null otherwise): r-tile rt only multiplies the k-blocks
  // kb_begin[rt] .. + kb_count[rt] (>= 1) -- the rows and columns of the operands are permuted so that the non-zero
  // blocks of S2 are contiguous -- and output row r of the permuted, padded row space goes to U row rowmap[r] (< 0: padding)
  const int* kb_begin;
  const int* kb_count;
  const int* rowmap;
};

__host__ __device__ inline int b_bytes(int NT) { return NT * BK * 2; }
__host__ __device__ inline int stage_bytes(int NT) { return 2 * A_BYTES + 2 * b_bytes(NT); }
inline size_t smem_bytes(int NT, int stages) {
  return 1024 /*alignment slack*/ + 1024 /*barriers*/ + (size_t)stages * stage_bytes(NT);
}

// SPARSE = false compiles the three tables away: the dense instantiations are the code they were before r02's
// block-sparse form (the row map inside the unrolled store loop cost the dense kernel 0.80 -> 0.99 ms when it was a
// run-time branch).
template <bool OUT_H, bool SPARSE = false, int EC = EPI_COLS>
__global__ void __launch_bounds__(NTHREADS, 1)
k_contract_h(const __grid_constant__ CUtensorMap tmVh, const __grid_constant__ CUtensorMap tmVl,
             const __grid_constant__ CUtensorMap tmSh, const __grid_constant__ CUtensorMap tmSl, const Params p) {
  using namespace ptx;
  pdl_launch_dependents();
  extern __shared__ unsigned char smem_raw[];
  const uint32_t raw_addr = smem_u32(smem_raw);
  const uint32_t base = (raw_addr + 1023u) & ~1023u;     // 1024-byte aligned: swizzle atoms
  unsigned char* sm = smem_raw + (base - raw_addr);
  // barrier block (first 1 KiB): full[8] empty[8] tmem_full[2] tmem_empty[2] tmem_slot
  const uint32_t bar_full = base, bar_empty = base + 64, bar_tfull = base + 128, bar_tempty = base + 144,
                 slot_addr = base + 160;
  volatile uint32_t* tmem_slot = reinterpret_cast<volatile uint32_t*>(sm + 160);
  const uint32_t tiles_addr = base + 1024;

  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const int nb = b_bytes(p.NT), sbytes = stage_bytes(p.NT);
  const int stages = p.stages;

  if (warp == 0 && lane == 0) {
    prefetch_tensormap(&tmVh);
    prefetch_tensormap(&tmVl);
    prefetch_tensormap(&tmSh);
    prefetch_tensormap(&tmSl);
  }
  if (warp == 1) {
    if (lane == 0) {
      for (int s = 0; s < MAX_STAGES; ++s) {
        mbar_init(bar_full + 8 * s, 1);
        mbar_init(bar_empty + 8 * s, 1);
      }
      for (int a = 0; a < 2; ++a) {
        mbar_init(bar_tfull + 8 * a, 1);
        mbar_init(bar_tempty + 8 * a, NUM_EPI_WARPS);
      }
      fence_barrier_init();
    }
    __syncwarp();
    tmem_alloc<1>(slot_addr, TMEM_COLS);
    tmem_relinquish<1>();
  }
  tc_fence_before();
  __syncthreads();
  tc_fence_after();
  const uint32_t tmem_base = *tmem_slot;
  pdl_wait();                     // everything above touches no global data: it overlaps the predecessor's tail

  const int cta = blockIdx.x, nctas = gridDim.x;
  const int tiles_per_plane = p.n_rt * p.t_tiles;

  if (warp == 0) {
    // ================================================================= TMA producer
    if (lane == 0) {
      int stage = 0;
      uint32_t phase = 0;
      for (int tile = cta; tile < p.total_tiles; tile += nctas) {
        const int pl = tile / tiles_per_plane, rem = tile - pl * tiles_per_plane;
        const int tt = rem / p.n_rt, rt = rem - tt * p.n_rt;
        const int t0 = tt * TM, r0 = rt * p.NT;
        const int k0 = SPARSE ? p.kb_begin[rt] : 0, kn = SPARSE ? p.kb_count[rt] : p.KB;
        for (int kb = k0; kb < k0 + kn; ++kb) {
          mbar_wait(bar_empty + 8 * stage, phase ^ 1u, 1);
          const uint32_t fb = bar_full + 8 * stage;
          const uint32_t sa = tiles_addr + stage * sbytes;
          mbar_arrive_expect_tx(fb, (uint32_t)(2 * A_BYTES + 2 * nb));
#pragma unroll
          for (int i = 0; i < TM / 64; ++i) {                     // 2 boxes of 64 t x BK q per operand half
            tma_load_3d(sa + i * (BK * 128), &tmVh, fb, t0 + 64 * i, kb * BK, p.plane0 + pl);
            tma_load_3d(sa + A_BYTES + i * (BK * 128), &tmVl, fb, t0 + 64 * i, kb * BK, p.plane0 + pl);
          }
          tma_load_2d(sa + 2 * A_BYTES, &tmSh, fb, kb * BK, r0);
          tma_load_2d(sa + 2 * A_BYTES + nb, &tmSl, fb, kb * BK, r0);
          if (++stage == stages) { stage = 0; phase ^= 1u; }
        }
      }
    }
  } else if (warp == 1) {
    // ================================================================= MMA issuer
    if (lane == 0) {
      // instruction descriptor: D fp32, A/B fp16, A MN-major, B K-major, N = NT, M = 128
      const uint32_t idesc = (1u << 4) | (1u << 15) | ((uint32_t)(p.NT >> 3) << 17) | ((uint32_t)(TM >> 4) << 24);
      int stage = 0, acc = 0;
      uint32_t phase = 0, acc_phase = 0;
      for (int tile = cta; tile < p.total_tiles; tile += nctas) {
        const int kn = SPARSE ? p.kb_count[tile % p.n_rt] : p.KB;   // r-tile index is the fastest tile coordinate
        for (int kb = 0, inchunk = 0; kb < kn; ++kb) {
          if (inchunk == 0) {                                      // new chunk: claim a TMEM accumulator
            mbar_wait(bar_tempty + 8 * acc, acc_phase ^ 1u, 2);
            tc_fence_after();
          }
          const uint32_t d = tmem_base + (uint32_t)(acc * ACC_COLS);
          mbar_wait(bar_full + 8 * stage, phase, 3);
          tc_fence_after();
          const uint32_t sa = tiles_addr + stage * sbytes;
          const uint64_t a_hi = make_smem_desc(sa, BK * 128, 1024, 2);
          const uint64_t a_lo = make_smem_desc(sa + A_BYTES, BK * 128, 1024, 2);
          const uint64_t b_hi = make_smem_desc(sa + 2 * A_BYTES, 16, 512, 4);
          const uint64_t b_lo = make_smem_desc(sa + 2 * A_BYTES + nb, 16, 512, 4);
#pragma unroll
          for (int kk = 0; kk < BK / 16; ++kk) {
            const uint64_t da = (uint64_t)(kk * (2048 >> 4));      // next 16 q of A: two 8-q groups
            const uint64_t db = (uint64_t)(kk * (32 >> 4));        // next 16 q of B: +32 B in the row
            mma_f16_ss<1>(d, a_hi + da, b_lo + db, idesc, (inchunk | kk) != 0 ? 1u : 0u);
            mma_f16_ss<1>(d, a_lo + da, b_hi + db, idesc, 1u);
            mma_f16_ss<1>(d, a_hi + da, b_hi + db, idesc, 1u);
          }
          mma_commit<1>(bar_empty + 8 * stage);
          if (++stage == stages) { stage = 0; phase ^= 1u; }
          if (++inchunk == p.kchunk || kb == kn - 1) {             // chunk complete: hand it to the epilogue
            mma_commit<1>(bar_tfull + 8 * acc);
            inchunk = 0;
            if (++acc == 2) { acc = 0; acc_phase ^= 1u; }
          }
        }
      }
    }
  } else {
    // ================================================================= epilogue: TMEM -> registers -> U[r][t]
    const int lg = warp & 3;                      // TMEM lane group this warp may read
    const int third = (warp - 2) >> 2;            // which slice of the NT columns
    const int cper = ((p.NT + 2) / 3 + 7) / 8 * 8;
    const int cbeg = third * cper;
    const int ncols = max(0, min(p.NT, cbeg + cper) - cbeg);       // multiple of 8, <= EC
    const float vb = *p.vbound;
    const float inv_sv = v_scale(p.bound_gain * vb, true);
    const float sz = OUT_H ? v_scale(p.zgain * vb, false) : 1.f;
    int acc = 0;
    uint32_t acc_phase = 0;
    float accr[EC];
    for (int tile = cta; tile < p.total_tiles; tile += nctas) {
      const int pl = tile / tiles_per_plane, rem = tile - pl * tiles_per_plane;
      const int tt = rem / p.n_rt, rt = rem - tt * p.n_rt;
      const int t = tt * TM + lg * 32 + lane;
#pragma unroll
      for (int i = 0; i < EC; ++i) accr[i] = 0.f;
      const int nchunks = ((SPARSE ? p.kb_count[rt] : p.KB) + p.kchunk - 1) / p.kchunk;
      for (int ch = 0; ch < nchunks; ++ch) {
        mbar_wait(bar_tfull + 8 * acc, acc_phase, 5);
        tc_fence_after();
        const uint32_t taddr = tmem_base + ((uint32_t)(lg * 32) << 16) + (uint32_t)(acc * ACC_COLS + cbeg);
        // EPI_ROUND groups of 8 columns in flight per wait (3 and 5 measured no faster: the drain is bound by the
        // tensor-memory read rate, not by the round trips)
#pragma unroll
        for (int g0 = 0; g0 < EC / 8; g0 += EPI_ROUND) {
          uint32_t v[EPI_ROUND][8];
#pragma unroll
          for (int g = g0; g < g0 + EPI_ROUND && g < EC / 8; ++g)
            if (g * 8 < ncols) tmem_ld_x8(taddr + g * 8, v[g - g0]);
          tmem_ld_wait();
#pragma unroll
          for (int g = g0; g < g0 + EPI_ROUND && g < EC / 8; ++g)
            if (g * 8 < ncols) {
#pragma unroll
              for (int c = 0; c < 8; ++c) accr[g * 8 + c] += __uint_as_float(v[g - g0][c]);
            }
        }
        tc_fence_before();
        __syncwarp();
        if (lane == 0) mbar_arrive(bar_tempty + 8 * acc);
        if (++acc == 2) { acc = 0; acc_phase ^= 1u; }
      }
      const int rbase = rt * p.NT + cbeg;
      const float* rs = p.rscale + rbase;
      if constexpr (OUT_H) {
        __half* Zh = p.Zh + (long long)pl * p.u_plane_stride + t;
        __half* Zl = Zh + (long long)p.Q * p.N;
#pragma unroll
        for (int c = 0; c < EC; ++c) {
          const int r = rbase + c;
          if (c < ncols && r < p.Q) {
            const float z = accr[c] * (rs[c] * inv_sv) * sz;
            const __half h = __float2half_rn(z);
            Zh[(long long)r * p.N] = h;
            Zl[(long long)r * p.N] = __float2half_rn(z - __half2float(h));
          }
        }
      } else {
        float* Uout = p.U + (long long)pl * p.u_plane_stride + t;
#pragma unroll
        for (int c = 0; c < EC; ++c) {
          const int r = rbase + c;
          if constexpr (SPARSE) {
            if (c < ncols) {
              const int rn = p.rowmap[r];
              if (rn >= 0) Uout[(long long)rn * p.N] = accr[c] * (rs[c] * inv_sv);
            }
          } else {
            if (c < ncols && r < p.Q) Uout[(long long)r * p.N] = accr[c] * (rs[c] * inv_sv);
          }
        }
      }
    }
  }

  // ------------------------------------------------------------------- teardown
  __syncwarp();
  tc_fence_before();
  __syncthreads();
  tc_fence_after();
  if (warp == 1) tmem_dealloc<1>(tmem_base, TMEM_COLS);
}

}  // namespace hc
}  // namespace gm
