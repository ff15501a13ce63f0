// a6 on tcgen05, "TS" form: the A operand (V_hi, V_lo) is read from TENSOR MEMORY instead of shared memory.
// Same contraction, orientation, split precision and two-level accumulation as gemm_tc.cuh; what changes:
//   * V tiles arrive by one un-swizzled TMA box [BK q][128 t] per k-block (no MMA reads them, so no
//     canonical layout is needed); converter thread t reads its BK samples down the q axis (conflict-free:
//     32 lanes = 32 consecutive t), splits them into V_hi / V_lo and writes both to tensor memory with
//     tcgen05.st (lane = t, one column per q) -- the K-major A layout the TS form requires.
//   * shared memory holds only raw V (8 KB) and S_hi, S_lo (2 x 13 KB) per stage: 6 stages instead of 5, no
//     V_lo tile, and the MMAs no longer read A from shared memory (about a quarter less traffic on the
//     shared-memory pipe, which ncu showed 71 % busy in the SS form).
//   * tensor memory: accumulators at columns [0, NT) and [NT, 2 NT), NT <= 208; the 96 columns above 416
//     hold three A stages of 32 columns (16 q of V_hi, 16 q of V_lo).
// Pipelines: smem ring (full: TMA -> converters; empty: MMA commit -> TMA), A ring in TMEM (conv: converters
// -> MMA; aempty: MMA commit -> converters), two accumulators (tmem_full / tmem_empty) drained per chunk.
#pragma once
#include "gemm_tc.cuh"

namespace gm {
namespace tc {

constexpr int TS_A_STAGES = 3;
constexpr int TS_A_COL0 = 416;

__host__ __device__ inline int ts_stage_bytes(int NT) { return A_BYTES + 2 * b_bytes(NT, 1); }
inline size_t ts_smem_bytes(int NT, int stages) { return 2048 + (size_t)stages * ts_stage_bytes(NT); }

__global__ void __launch_bounds__(NTHREADS, 1)
k_contract_ts(const __grid_constant__ CUtensorMap tmV, const __grid_constant__ CUtensorMap tmShi,
              const __grid_constant__ CUtensorMap tmSlo, const Params p) {
  using namespace ptx;
  extern __shared__ unsigned char smem_raw[];
  const uint32_t raw_addr = smem_u32(smem_raw);
  const uint32_t base = (raw_addr + 1023u) & ~1023u;
  unsigned char* sm = smem_raw + (base - raw_addr);
  // barrier block: full[8] empty[8] conv[4] aempty[4] tmem_full[2] tmem_empty[2] tmem_slot
  const uint32_t bar_full = base, bar_empty = base + 64, bar_conv = base + 128, bar_aempty = base + 160,
                 bar_tfull = base + 192, bar_tempty = base + 208, slot_addr = base + 224;
  volatile uint32_t* tmem_slot = reinterpret_cast<volatile uint32_t*>(sm + 224);
  const uint32_t tiles_addr = base + 1024;
  unsigned char* tiles_ptr = sm + 1024;

  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const int nb = b_bytes(p.NT, 1), sbytes = ts_stage_bytes(p.NT);
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
      }
      for (int s = 0; s < TS_A_STAGES; ++s) {
        mbar_init(bar_conv + 8 * s, 4);
        mbar_init(bar_aempty + 8 * s, 1);
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

  const int first = blockIdx.x, step = gridDim.x;
  const int tiles_per_plane = p.n_rt * p.t_tiles;

  if (warp == 0) {
    // ================================================================= TMA producer
    if (lane == 0) {
      int stage = 0;
      uint32_t phase = 0;
      const uint32_t tx = (uint32_t)(A_BYTES + 2 * nb);
      for (int tile = first; tile < p.total_tiles; tile += step) {
        const int pl = tile / tiles_per_plane, rem = tile - pl * tiles_per_plane;
        const int tt = rem / p.n_rt, rt = rem - tt * p.n_rt;
        for (int kb = 0; kb < p.KB; ++kb) {
          mbar_wait(bar_empty + 8 * stage, phase ^ 1u, 1);
          const uint32_t fb = bar_full + 8 * stage;
          const uint32_t sa = tiles_addr + stage * sbytes;
          mbar_arrive_expect_tx(fb, tx);
          tma_load_3d(sa, &tmV, fb, tt * TM, kb * BK, p.plane0 + pl);              // [BK q][128 t], no swizzle
          tma_load_2d(sa + A_BYTES, &tmShi, fb, kb * BK, rt * p.NT);
          tma_load_2d(sa + A_BYTES + nb, &tmSlo, fb, kb * BK, rt * p.NT);
          if (++stage == stages) { stage = 0; phase ^= 1u; }
        }
      }
    }
  } else if (warp == 1) {
    // ================================================================= MMA issuer
    if (lane == 0) {
      // D fp32, A/B tf32, A K-major (tensor memory), B K-major, N = NT, M = 128
      const uint32_t idesc = (1u << 4) | (2u << 7) | (2u << 10) | ((uint32_t)(p.NT >> 3) << 17) |
                             ((uint32_t)(TM >> 4) << 24);
      int stage = 0, ts = 0, acc = 0;
      uint32_t ts_phase = 0, acc_phase = 0;
      for (int tile = first; tile < p.total_tiles; tile += step) {
        for (int kb = 0, inchunk = 0; kb < p.KB; ++kb) {
          if (inchunk == 0) {
            mbar_wait(bar_tempty + 8 * acc, acc_phase ^ 1u, 2);
            tc_fence_after();
          }
          const uint32_t d = tmem_base + (uint32_t)(acc * p.NT);
          mbar_wait(bar_conv + 8 * ts, ts_phase, 3);       // A stage written (implies the smem stage has landed)
          tc_fence_after();
          const uint32_t sa = tiles_addr + stage * sbytes;
          const uint32_t a_hi = tmem_base + (uint32_t)(TS_A_COL0 + ts * 2 * BK), a_lo = a_hi + BK;
          const uint64_t b_hi = make_smem_desc(sa + A_BYTES, 16, B_SBO, B_LAYOUT);
          const uint64_t b_lo = make_smem_desc(sa + A_BYTES + nb, 16, B_SBO, B_LAYOUT);
#pragma unroll
          for (int kk = 0; kk < BK / 8; ++kk) {
            const uint64_t db = (uint64_t)(kk * (32 >> 4));
            mma_tf32_ts<1>(d, a_hi + kk * 8, b_lo + db, idesc, (inchunk | kk) != 0 ? 1u : 0u);
            mma_tf32_ts<1>(d, a_lo + kk * 8, b_hi + db, idesc, 1u);
            mma_tf32_ts<1>(d, a_hi + kk * 8, b_hi + db, idesc, 1u);
          }
          mma_commit<1>(bar_empty + 8 * stage);            // smem stage free
          mma_commit<1>(bar_aempty + 8 * ts);              // A stage in tensor memory free
          if (++stage == stages) stage = 0;
          if (++ts == TS_A_STAGES) { ts = 0; ts_phase ^= 1u; }
          if (++inchunk == p.kchunk || kb == p.KB - 1) {
            mma_commit<1>(bar_tfull + 8 * acc);
            inchunk = 0;
            if (++acc == 2) { acc = 0; acc_phase ^= 1u; }
          }
        }
      }
    }
  } else if (warp < 6) {
    // ================================================================= converters: smem V -> TMEM V_hi, V_lo
    const int lg = warp & 3;                       // TMEM lane group this warp may write
    const int tl = lg * 32 + lane;                 // time sample within the tile
    int stage = 0, ts = 0;
    uint32_t phase = 0, ts_phase = 0;
    for (int tile = first; tile < p.total_tiles; tile += step) {
      for (int kb = 0; kb < p.KB; ++kb) {
        mbar_wait(bar_full + 8 * stage, phase, 4);
        const float* raw = reinterpret_cast<const float*>(tiles_ptr + (size_t)stage * sbytes) + tl;
        uint32_t vh[BK], vl[BK];
#pragma unroll
        for (int q = 0; q < BK; ++q) {
          const float v = raw[q * TM];
          const uint32_t h = __float_as_uint(v) & 0xFFFFE000u;
          vh[q] = h;
          vl[q] = __float_as_uint(to_tf32_rna(v - __uint_as_float(h)));
        }
        mbar_wait(bar_aempty + 8 * ts, ts_phase ^ 1u, 6);
        tc_fence_after();
        const uint32_t taddr = tmem_base + ((uint32_t)(lg * 32) << 16) + (uint32_t)(TS_A_COL0 + ts * 2 * BK);
        tmem_st_x16(taddr, vh);
        tmem_st_x16(taddr + BK, vl);
        tmem_st_wait();
        tc_fence_before();
        __syncwarp();
        if (lane == 0) mbar_arrive(bar_conv + 8 * ts);
        if (++stage == stages) { stage = 0; phase ^= 1u; }
        if (++ts == TS_A_STAGES) { ts = 0; ts_phase ^= 1u; }
      }
    }
  } else {
    // ================================================================= epilogue: TMEM -> registers -> U[r][t]
    const int lg = warp & 3;
    const int third = (warp - 6) >> 2;
    const int cper = ((p.NT + 2) / 3 + 7) / 8 * 8;
    const int cbeg = third * cper;
    const int ncols = max(0, min(p.NT, cbeg + cper) - cbeg);
    const int nchunks = (p.KB + p.kchunk - 1) / p.kchunk;
    int acc = 0;
    uint32_t acc_phase = 0;
    float accr[EPI_COLS];
    for (int tile = first; tile < p.total_tiles; tile += step) {
      const int pl = tile / tiles_per_plane, rem = tile - pl * tiles_per_plane;
      const int tt = rem / p.n_rt, rt = rem - tt * p.n_rt;
      const int t = tt * TM + lg * 32 + lane;
      float* Uout = p.U + (long long)pl * p.u_plane_stride + t;
#pragma unroll
      for (int i = 0; i < EPI_COLS; ++i) accr[i] = 0.f;
      for (int ch = 0; ch < nchunks; ++ch) {
        mbar_wait(bar_tfull + 8 * acc, acc_phase, 5);
        tc_fence_after();
        const uint32_t taddr = tmem_base + ((uint32_t)(lg * 32) << 16) + (uint32_t)(acc * p.NT + cbeg);
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

  __syncwarp();
  tc_fence_before();
  __syncthreads();
  tc_fence_after();
  if (warp == 1) tmem_dealloc<1>(tmem_base, TMEM_COLS);
}

}  // namespace tc
}  // namespace gm
