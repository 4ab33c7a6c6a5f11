// mma_pipeline.cuh — the FP64 tensor-core mainloop shared by the transform GEMMs and the fused pair kernel.
//
// Both operands are "K-major": row r of an operand holds its K values contiguously in global memory.
// One pipeline stage holds a K-block of 8 doubles for TM rows of operand A and TN rows of operand B,
// each stored densely as [row][8] (64 B per row).  A dedicated producer warp fills stages with TMA
// (cp.async.bulk.tensor, box {8, rows...}); completion is signalled on a "full" mbarrier; consumer
// warps release a stage by arriving on its "empty" mbarrier.
//
// Consumer fragment loads: lane (g,t) reads the 16-byte pair (k=2t, 2t+1) of row g with one LDS.128.
// A quarter-warp (g in {0,1}, t in 0..3) therefore reads 128 contiguous bytes: conflict-free without
// padding or swizzle.  The two doubles feed two DMMA.8x8x4: the first covers k in {0,2,4,6}, the second
// k in {1,3,5,7}; A and B use the same permutation, so the sum over the K-block is unchanged.
// Measured on B200 (profiles/fp64_peak_r01.md): this smem->DMMA loop sustains 36.96 of 37.15 TFLOP/s.
#pragma once

#include "sie_common.cuh"

namespace sie {

template <int WM_, int WN_, int NWM_, int NWN_, int STAGES_>
struct TileCfg {
    static constexpr int WM = WM_, WN = WN_, NWM = NWM_, NWN = NWN_, STAGES = STAGES_;
    static constexpr int TM = WM * NWM, TN = WN * NWN;  // CTA tile
    static constexpr int MT = WM / 8, NT = WN / 8;      // DMMA tiles per warp
    static constexpr int NCONS = NWM * NWN;             // consumer warps
    static constexpr int NTHREADS = (NCONS + 1) * 32;   // + one producer warp
    static constexpr int KB = 8;                        // K-block (doubles) per stage
    static constexpr int STAGE_DOUBLES = (TM + TN) * KB;
    static constexpr int STAGE_BYTES = STAGE_DOUBLES * 8;
    static_assert(WM % 8 == 0 && WN % 8 == 0, "warp tile must be a multiple of the 8x8 DMMA tile");
};

struct PipeState {
    int stage = 0;
    uint32_t phase = 0;
    template <int STAGES>
    __device__ __forceinline__ void advance() {
        if (++stage == STAGES) {
            stage = 0;
            phase ^= 1u;
        }
    }
};

// Consumer side: accumulate `kblocks` K-blocks into acc (zeroed here).
template <class Cfg>
__device__ __forceinline__ void consume_tile(double (&acc)[Cfg::MT][Cfg::NT][2], const double* __restrict__ stages,
                                             uint64_t* full, uint64_t* empty, int kblocks, PipeState& ps, int wm, int wn,
                                             int lane) {
    const int g = lane >> 2, t = lane & 3;
#pragma unroll
    for (int i = 0; i < Cfg::MT; ++i)
#pragma unroll
        for (int j = 0; j < Cfg::NT; ++j) {
            acc[i][j][0] = 0.0;
            acc[i][j][1] = 0.0;
        }
    const int offA = (wm * Cfg::WM + g) * Cfg::KB + 2 * t;
    const int offB = Cfg::TM * Cfg::KB + (wn * Cfg::WN + g) * Cfg::KB + 2 * t;
    for (int kb = 0; kb < kblocks; ++kb) {
        mbar_wait(&full[ps.stage], ps.phase);
        const double* s = stages + ps.stage * Cfg::STAGE_DOUBLES;
        double2 a[Cfg::MT], b[Cfg::NT];
#pragma unroll
        for (int i = 0; i < Cfg::MT; ++i) a[i] = *reinterpret_cast<const double2*>(s + offA + i * 8 * Cfg::KB);
#pragma unroll
        for (int j = 0; j < Cfg::NT; ++j) b[j] = *reinterpret_cast<const double2*>(s + offB + j * 8 * Cfg::KB);
#pragma unroll
        for (int i = 0; i < Cfg::MT; ++i)
#pragma unroll
            for (int j = 0; j < Cfg::NT; ++j) {
                dmma884(acc[i][j][0], acc[i][j][1], a[i].x, b[j].x);
                dmma884(acc[i][j][0], acc[i][j][1], a[i].y, b[j].y);
            }
        __syncwarp();
        if (lane == 0) mbar_arrive(&empty[ps.stage]);
        ps.advance<Cfg::STAGES>();
    }
}

// Producer side (one elected lane): stream `kblocks` K-blocks of two operand tiles.
//   operand A tile: box at coordinates (k, a1, a2) of mapA -> first TM rows of the stage
//   operand B tile: box at coordinates (k, b1, b2) of mapB -> next TN rows
// tx_bytes = bytes of both boxes (TMA counts the full box even where it zero-fills out of bounds).
template <class Cfg>
__device__ __forceinline__ void produce_tile(double* stages, uint64_t* full, uint64_t* empty, int kblocks, PipeState& ps,
                                             const CUtensorMap* mapA, int a1, int a2, const CUtensorMap* mapB, int b1, int b2,
                                             uint32_t tx_bytes) {
    for (int kb = 0; kb < kblocks; ++kb) {
        mbar_wait(&empty[ps.stage], ps.phase ^ 1u);
        double* s = stages + ps.stage * Cfg::STAGE_DOUBLES;
        mbar_arrive_expect_tx(&full[ps.stage], tx_bytes);
        tma_load_3d(s, mapA, &full[ps.stage], kb * Cfg::KB, a1, a2);
        tma_load_3d(s + Cfg::TM * Cfg::KB, mapB, &full[ps.stage], kb * Cfg::KB, b1, b2);
        ps.advance<Cfg::STAGES>();
    }
}

template <class Cfg>
__device__ __forceinline__ void pipeline_init(uint64_t* full, uint64_t* empty, int tid) {
    if (tid == 0) {
#pragma unroll
        for (int s = 0; s < Cfg::STAGES; ++s) {
            mbar_init(&full[s], 1);
            mbar_init(&empty[s], Cfg::NCONS);
        }
        fence_mbar_init();
    }
}

}  // namespace sie
