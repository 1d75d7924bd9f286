// tuning.h -- the shipped kernel configurations (tile sizes, ring depths, CTAs per SM), as measured
// on B200 (profiles/r01_sweeps.md, profiles/r02_*.md).  Plain compile-time tables: both the create
// calls (tile tables, shapes) and the launch code read them, nothing else decides a kernel shape.
#pragma once

#include <cuda_runtime.h>

#include "../../include/msolve.h"

namespace msolve {

// TMA-staged BSR3 kernel: block rows per tile, ring depth, CTAs per SM.  Many small CTAs per SM
// (independent tiles in flight hide the x-gather latency), a 2-deep ring is enough for the bulk
// copies, and a small shared-memory footprint leaves L1 for the gathers.
template <typename E> struct BsrTile;
template <> struct BsrTile<double2> { static constexpr int TB = 12, STAGES = 2, CPS = 5; };
template <> struct BsrTile<float2>  { static constexpr int TB = 24, STAGES = 2, CPS = 4; };
// the second BiCGStab-M SpMV carries five fp64 accumulators: one CTA per SM less keeps it from spilling
constexpr int kBsrCpsLessB2 = 1;

// Matrix-free lattice operator.  (term, site) kernel k_spmv_lat_tma: sites per tile, ring depth, CTAs per SM.
template <typename E> struct LatTile;
template <> struct LatTile<double2> { static constexpr int NS = 32, STAGES = 2, CPS = 2; };
template <> struct LatTile<float2>  { static constexpr int NS = 32, STAGES = 2, CPS = 4; };
// warp-per-tile all-TMA kernel k_spmv_lat_warp: consumer warps, ring depth; producer warps (bulk-copy issue is its
// bottleneck: 1 producer 0.47 ms, 2: 0.25 ms, 4: 0.150 ms on config 4 complex64)
template <typename E> struct LatWarpTile;
template <> struct LatWarpTile<double2> { static constexpr int W = 2, STAGES = 4; };
template <> struct LatWarpTile<float2>  { static constexpr int W = 4, STAGES = 8; };
constexpr int kLatWarpProducers = 4;
// hybrid kernel k_spmv_lat_hyb: consumer warps and ring depth (a bigger ring takes the L1 the gathers need)
template <typename E> struct LatHybTile;
template <> struct LatHybTile<double2> { static constexpr int W = 6, STAGES = 6; };
template <> struct LatHybTile<float2>  { static constexpr int W = 8, STAGES = 8; };
// blocked kernel k_spmv_lat_blk: block of R1 x R2 x0-rows per tile, ring depth (= producer warps); the stage of a
// 2 x 2 block is 70.7 KB in complex64 (three fit), 141 KB in complex128 (hence 2 x 1 there: 78.3 KB, two stages)
template <typename E> struct LatBlkTile;
template <> struct LatBlkTile<double2> { static constexpr int R1 = 2, R2 = 1, STAGES = 2; };
template <> struct LatBlkTile<float2>  { static constexpr int R1 = 2, R2 = 2, STAGES = 3; };
// default lattice tile kernel per element type where the blocked kernel does not apply (MSOLVE_CFG_LATTICE_KERNEL = 0):
// 1 = (term, site), 2 = warp, 3 = hybrid
template <typename E> struct LatDefault;
template <> struct LatDefault<double2> { static constexpr int kernel = 3; };   // 0.238 ms (all-TMA 0.269 / 0.277)
template <> struct LatDefault<float2>  { static constexpr int kernel = 2; };   // 0.149 ms (hybrid 0.168)

// Merge-path CSR: tile capacity (non-zeros), ring depth (>= 3: the consumers wait for tile t+1 before they work
// on tile t), CTAs per SM.
template <typename E> struct MergeTile { static constexpr int CAP = 2048, STAGES = 3, CPS = 2; };
template <> struct MergeTile<double2> { static constexpr int CAP = 1024, STAGES = 4, CPS = 2; };

// TMA-staged vector-CSR: ring depth and CTAs per SM; lanes per row and non-zeros per lane are chosen per matrix
// at create time (csr_tile_shape).  Config 4 as CSR: complex128 8 lanes x 4, 3 stages, 5 CTAs per SM: 0.559 ms
// (vector kernel 0.874); complex64 4 lanes x 8: 0.324 ms.
template <typename E> struct CsrTile { static constexpr int STAGES = 3, CPS = 5; };

// Fused multishift updates: shifts in flight per thread (2 * UNR independent 16-byte loads on top of r and Ap);
// 4 is the measured optimum for both k_cgm_update and k_bi_update.
constexpr int kUnrollCgm = 4, kUnrollBi = 4;
// shifts in flight per thread in the flush of the deferred update (on top of the chunk's residuals in registers)
constexpr int kUnrollFlush = 2;
// TMA-staged CG-M update: ring depth, and how many items later a stage is handed back
constexpr int kUpdStages = 6, kUpdLag = 2;

}  // namespace msolve
