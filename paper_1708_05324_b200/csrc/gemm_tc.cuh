// a6 on the 5th-generation tensor cores: U[j][r][t] = sum_q S2[r][q] V[j][q][t]  (the
// sum over m,n of Eq. 1 -- "by a large margin the most computationally expensive")
// as a split-precision ("3xTF32") tcgen05 GEMM with fp32 accumulation in tensor memory.
//
// Orientation: D[t][r] = sum_q A[t][q] B[r][q] with A = V_j^T and B = S2.
//   * M = t: 128 samples per CTA -- N is a power of two, so
//     the M tiles have no ragged edge; each TMEM lane is one time sample, so the epilogue's stores
//     (one column r at a time, 32 lanes = 32 consecutive t) are coalesced into U[r][t].
//   * N = r: NT packed pair rows per tile, NT = 16-multiple <= 256 chosen so that n_rt*NT >= Q with
//     < 2 % padding (Q = 1035 -> 5 x 208).
//   * K = q: BK = 16 per k-block (a 64-byte swizzle row of S2), 2 MMAs of K = 8 per product; the small
//     k-block lets 5 stages (43 KB each) fit in shared memory: with BK = 32 only 2 fit and the MMA pipe
//     starved on TMA latency (measured 1.58 ms against a 1.06 ms MMA-only floor at config 5).
//   A is "MN-major" (t contiguous in V[q][t]) in the 32-byte-atom 128-byte swizzle, the one MN-major
//   layout kind::tf32 accepts; B is K-major (q contiguous in S2[r][q]) in the plain 128-byte swizzle.
//
// Split precision: the tensor core reads fp32 words as TF32 and ignores the low 13 mantissa bits
// (measured: masking them first changes nothing).
//   V = V_hi + V_lo,  V_hi = V with the low 13 bits cleared (what the MMA sees when fed raw V),
//                     V_lo = tf32_rna(V - V_hi)   -- formed in shared memory by 4 converter warps;
//   S2 = S_hi + S_lo, both rounded to TF32 on the host at plan time (fp64 source);
//   D += V_hi S_lo + V_lo S_hi + V_hi S_hi   (the dropped V_lo S_lo term is 2^-22 relative).
// Two-level accumulation: the tensor core's fp32 accumulate truncates, which biases a long sum (measured
// on B200: relative error 8e-7 at K = 120, 7e-6 at K = 1035, linear in K).  So a TMEM accumulator only
// ever holds `kchunk` k-blocks; the epilogue warps drain each chunk into fp32 registers with
// round-to-nearest adds while the MMAs of the next chunk fill the other TMEM accumulator.
//
// Warp roles (576 threads): warp 0 TMA producer, warp 1 MMA issuer + TMEM allocator, warps 2-5
// converters, warps 6-17 epilogue (three per TMEM lane group, each owning a third of the NT columns).
// Pipelines: smem stages (full -> conv -> empty) and two TMEM accumulators (tmem_full / tmem_empty).
#pragma once
#include <cuda.h>

#include "cx.cuh"
#include "ptx_sm100.cuh"

namespace gm {
namespace tc {

constexpr int BK = 16;                                  // q per k-block (16: 5 smem stages fit; 32: only 2)
constexpr int B_LAYOUT = BK == 32 ? 2 : 4;              // smem descriptor layout type of B: SWIZZLE_128B / SWIZZLE_64B
constexpr int B_SBO = 8 * BK * 4;                       // bytes between 8-row groups of B
constexpr int TM = 128;                                 // t per CTA
constexpr int NUM_EPI_WARPS = 12;                       // 3 per TMEM lane group
constexpr int NTHREADS = 32 * (6 + NUM_EPI_WARPS);      // 576
constexpr int EPI_COLS = 72;                            // max columns one epilogue warp accumulates
constexpr int A_BYTES = TM * BK * 4;                    // 16 KiB: one A tile (raw or lo)
constexpr int MAX_STAGES = 8;
constexpr int TMEM_COLS = 512;
constexpr int ACC_COLS = 256;                           // column stride between the two accumulators

struct Params {
  float* U;                    // [plane][Q][N]
  long long u_plane_stride;    // elements
  int Q, N, NT, KB, n_rt, t_tiles, total_tiles, plane0, stages, kchunk;
};

__host__ __device__ inline int b_bytes(int NT) { return NT * BK * 4; }
__host__ __device__ inline int stage_bytes(int NT) { return 2 * A_BYTES + 2 * b_bytes(NT); }
inline size_t smem_bytes(int NT, int stages) {
  return 1024 /*alignment slack*/ + 1024 /*barriers*/ + (size_t)stages * stage_bytes(NT);
}

__global__ void __launch_bounds__(NTHREADS, 1)
k_contract_tc(const __grid_constant__ CUtensorMap tmV, const __grid_constant__ CUtensorMap tmShi,
              const __grid_constant__ CUtensorMap tmSlo, const Params p) {
  using namespace ptx;
  pdl_launch_dependents();
  extern __shared__ unsigned char smem_raw[];
  const uint32_t raw_addr = smem_u32(smem_raw);
  const uint32_t base = (raw_addr + 1023u) & ~1023u;     // 1024-byte aligned: swizzle atoms
  unsigned char* sm = smem_raw + (base - raw_addr);
  // barrier block (first 1 KiB): full[8] empty[8] conv[8] tmem_full[2] tmem_empty[2] tmem_slot
  const uint32_t bar_full = base, bar_empty = base + 64, bar_conv = base + 128, bar_tfull = base + 192,
                 bar_tempty = base + 208, slot_addr = base + 224;
  volatile uint32_t* tmem_slot = reinterpret_cast<volatile uint32_t*>(sm + 224);
  const uint32_t tiles_addr = base + 1024;
  unsigned char* tiles_ptr = sm + 1024;

  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const int nb = b_bytes(p.NT), sbytes = stage_bytes(p.NT);
  const int stages = p.stages;

  if (warp == 0 && lane == 0) {
    prefetch_tensormap(&tmV);
    prefetch_tensormap(&tmShi);
    prefetch_tensormap(&tmSlo);
  }
  if (warp == 1) {
    if (lane == 0) {
      for (int s = 0; s < MAX_STAGES; ++s) {
        mbar_init(bar_full + 8 * s, 1);
        mbar_init(bar_empty + 8 * s, 1);
        mbar_init(bar_conv + 8 * s, 4);
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

  const int pair = blockIdx.x, npairs = gridDim.x;
  const int tiles_per_plane = p.n_rt * p.t_tiles;

  if (warp == 0) {
    // ================================================================= TMA producer
    if (lane == 0) {
      int stage = 0;
      uint32_t phase = 0;
      for (int tile = pair; tile < p.total_tiles; tile += npairs) {
        const int pl = tile / tiles_per_plane, rem = tile - pl * tiles_per_plane;
        const int tt = rem / p.n_rt, rt = rem - tt * p.n_rt;
        const int t0 = tt * TM;
        const int r0 = rt * p.NT;
        for (int kb = 0; kb < p.KB; ++kb) {
          mbar_wait(bar_empty + 8 * stage, phase ^ 1u, 1);
          const uint32_t fb = bar_full + 8 * stage;
          const uint32_t sa = tiles_addr + stage * sbytes;
          mbar_arrive_expect_tx(fb, (uint32_t)(A_BYTES + 2 * nb));
#pragma unroll
          for (int i = 0; i < TM / 32; ++i)                       // 4 boxes of 32 t x BK q
            tma_load_3d(sa + i * (BK * 128), &tmV, fb, t0 + 32 * i, kb * BK, p.plane0 + pl);
          tma_load_2d(sa + 2 * A_BYTES, &tmShi, fb, kb * BK, r0);
          tma_load_2d(sa + 2 * A_BYTES + nb, &tmSlo, fb, kb * BK, r0);
          if (++stage == stages) { stage = 0; phase ^= 1u; }
        }
      }
    }
  } else if (warp == 1) {
    // ================================================================= MMA issuer
    if (lane == 0) {
      // instruction descriptor: D fp32, A/B tf32, A MN-major, B K-major, N = NT, M = 128
      const uint32_t idesc = (1u << 4) | (2u << 7) | (2u << 10) | (1u << 15) | ((uint32_t)(p.NT >> 3) << 17) |
                             ((uint32_t)(TM >> 4) << 24);
      int stage = 0, acc = 0;
      uint32_t phase = 0, acc_phase = 0;
      for (int tile = pair; tile < p.total_tiles; tile += npairs) {
        for (int kb = 0, inchunk = 0; kb < p.KB; ++kb) {
          if (inchunk == 0) {                                      // new chunk: claim a TMEM accumulator
            mbar_wait(bar_tempty + 8 * acc, acc_phase ^ 1u, 2);
            tc_fence_after();
          }
          const uint32_t d = tmem_base + (uint32_t)(acc * ACC_COLS);
          mbar_wait(bar_conv + 8 * stage, phase, 3);
          tc_fence_after();
          const uint32_t sa = tiles_addr + stage * sbytes;
          // A: MN-major, 128-byte swizzle with 32-byte atoms (TMA SWIZZLE_128B_ATOM_32B): rows of 32 t
          // (128 B) per q, 4-q groups 512 B apart (SBO), 32-t groups BK*128 B apart (LBO)
          const uint64_t a_raw = make_smem_desc(sa, BK * 128, 512, 1);
          const uint64_t a_lo = make_smem_desc(sa + A_BYTES, BK * 128, 512, 1);
          // B: K-major rows of BK q (64 B: SWIZZLE_64B), 8-row groups B_SBO apart; LBO unused when swizzled
          const uint64_t b_hi = make_smem_desc(sa + 2 * A_BYTES, 16, B_SBO, B_LAYOUT);
          const uint64_t b_lo = make_smem_desc(sa + 2 * A_BYTES + nb, 16, B_SBO, B_LAYOUT);
#pragma unroll
          for (int kk = 0; kk < BK / 8; ++kk) {
            const uint64_t da = (uint64_t)(kk * (1024 >> 4));      // next 8 q of A: +1024 B
            const uint64_t db = (uint64_t)(kk * (32 >> 4));        // next 8 q of B: +32 B in the row
            mma_tf32_ss<1>(d, a_raw + da, b_lo + db, idesc, (inchunk | kk) != 0 ? 1u : 0u);
            mma_tf32_ss<1>(d, a_lo + da, b_hi + db, idesc, 1u);
            mma_tf32_ss<1>(d, a_raw + da, b_hi + db, idesc, 1u);
          }
          mma_commit<1>(bar_empty + 8 * stage);
          if (++stage == stages) { stage = 0; phase ^= 1u; }
          if (++inchunk == p.kchunk || kb == p.KB - 1) {           // chunk complete: hand it to the epilogue
            mma_commit<1>(bar_tfull + 8 * acc);
            inchunk = 0;
            if (++acc == 2) { acc = 0; acc_phase ^= 1u; }
          }
        }
      }
    }
  } else if (warp < 6) {
    // ================================================================= converters: V_lo (and V_hi)
    const int tid_c = threadIdx.x - 64;
    int stage = 0;
    uint32_t phase = 0;
    for (int tile = pair; tile < p.total_tiles; tile += npairs) {
      for (int kb = 0; kb < p.KB; ++kb) {
        mbar_wait(bar_full + 8 * stage, phase, 4);
        float4* raw = reinterpret_cast<float4*>(tiles_ptr + (size_t)stage * sbytes);
        float4* lo = reinterpret_cast<float4*>(tiles_ptr + (size_t)stage * sbytes + A_BYTES);
#pragma unroll
        for (int j = 0; j < A_BYTES / 16 / 128; ++j) {
          const int idx = tid_c + 128 * j;
          const float4 v = raw[idx];
          float4 h, l;
          h.x = __uint_as_float(__float_as_uint(v.x) & 0xFFFFE000u);
          h.y = __uint_as_float(__float_as_uint(v.y) & 0xFFFFE000u);
          h.z = __uint_as_float(__float_as_uint(v.z) & 0xFFFFE000u);
          h.w = __uint_as_float(__float_as_uint(v.w) & 0xFFFFE000u);
          l.x = to_tf32_rna(v.x - h.x);
          l.y = to_tf32_rna(v.y - h.y);
          l.z = to_tf32_rna(v.z - h.z);
          l.w = to_tf32_rna(v.w - h.w);
          lo[idx] = l;
        }
        fence_proxy_async_smem();                 // generic-proxy writes -> visible to the MMA's async reads
        __syncwarp();
        if (lane == 0) mbar_arrive(bar_conv + 8 * stage);
        if (++stage == stages) { stage = 0; phase ^= 1u; }
      }
    }
  } else {
    // ================================================================= epilogue: TMEM -> registers -> U[r][t]
    const int lg = warp & 3;                      // TMEM lane group this warp may read
    const int third = (warp - 6) >> 2;            // which slice of the NT columns
    const int cper = ((p.NT + 2) / 3 + 7) / 8 * 8;
    const int cbeg = third * cper;
    const int ncols = max(0, min(p.NT, cbeg + cper) - cbeg);       // multiple of 8, <= EPI_COLS
    const int nchunks = (p.KB + p.kchunk - 1) / p.kchunk;
    int acc = 0;
    uint32_t acc_phase = 0;
    float accr[EPI_COLS];
    for (int tile = pair; tile < p.total_tiles; tile += npairs) {
      const int pl = tile / tiles_per_plane, rem = tile - pl * tiles_per_plane;
      const int tt = rem / p.n_rt, rt = rem - tt * p.n_rt;
      const int t = tt * TM + lg * 32 + lane;
      float* Uout = p.U + (long long)pl * p.u_plane_stride + t;
#pragma unroll
      for (int i = 0; i < EPI_COLS; ++i) accr[i] = 0.f;
      for (int ch = 0; ch < nchunks; ++ch) {
        mbar_wait(bar_tfull + 8 * acc, acc_phase, 5);
        tc_fence_after();
        const uint32_t taddr = tmem_base + ((uint32_t)(lg * 32) << 16) + (uint32_t)(acc * ACC_COLS + cbeg);
#pragma unroll
        for (int g = 0; g < EPI_COLS / 8; g += 2) {
          if (g * 8 < ncols) {
            uint32_t v0[8], v1[8];
            tmem_ld_x8(taddr + g * 8, v0);
            const bool two = (g + 1) * 8 < ncols;
            if (two) tmem_ld_x8(taddr + (g + 1) * 8, v1);
            tmem_ld_wait();
#pragma unroll
            for (int c = 0; c < 8; ++c) accr[g * 8 + c] += __uint_as_float(v0[c]);
            if (two) {
#pragma unroll
              for (int c = 0; c < 8; ++c) accr[(g + 1) * 8 + c] += __uint_as_float(v1[c]);
            }
          }
        }
        tc_fence_before();
        __syncwarp();
        if (lane == 0) mbar_arrive(bar_tempty + 8 * acc);
        if (++acc == 2) { acc = 0; acc_phase ^= 1u; }
      }
      const int rbase = rt * p.NT + cbeg;
#pragma unroll
      for (int c = 0; c < EPI_COLS; ++c) {
        const int r = rbase + c;
        if (c < ncols && r < p.Q) Uout[(long long)r * p.N] = accr[c];
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

}  // namespace tc
}  // namespace gm
