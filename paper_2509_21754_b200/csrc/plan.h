// plan.h -- host-only launch planning for the FITrig library (no CUDA types here).
#pragma once
#include <stdint.h>

#include "fitrig.h"

namespace fitrig {

constexpr int kFastTile = 32;          // pixel block edge of the fused path = the paper's default tile
constexpr int kTileBytes = 32 * 32 * 4;  // one 32x32 fp32 block
constexpr int kMaxSmemPerCta = 227 * 1024;
constexpr int kMaxTilesPerBox = 8;     // fused path: tiles per TMA box (256 columns, the TMA box limit) = consumer warps per CTA
constexpr int kMaxStages = 8;          // fused path: deepest ring of boxes
constexpr int kMinUnitsPerCta = 2;     // fused path: fewest (box column, unit) pairs worth a CTA of its own
constexpr int kMaxAccAsync = 8;        // accumulations up to this length re-read their arg-max pixels with cp.async
constexpr int kScratchRec = 3 * kMaxAccAsync;  // fused kernel scratch: [0, kScratchRec) re-read pixels, then 2 records
constexpr int kScratchVec = kScratchRec + 2;   // float4 per warp of arg-max scratch (fused kernel)

struct NormParams {  // fitrig_params with defaults applied
  int tile;
  float C;
  int ref_mode;
  float M_override;
  int branch;
  int strip_rows;
  int device;
  int row_offset;
  int accumulate;  // >= 1
  int harmonics;   // 1, 2, 4, .., 32
  int stride;      // window stride in pixels; == tile: the paper's non-overlapping tiles
  int batch;       // >= 1 independent stacks per call
};

// Debug / tuning switches, read from the environment ONCE per fitrig_create / fitrig_plan_query call (documented in
// include/fitrig.h); 0 = not set.
struct Tuning {
  int box_tiles;        // FITRIG_BOX_TILES      fused path: adjacent 32x32 blocks per TMA box (1..8)
  int stages;           // FITRIG_STAGES         fused path: ring depth
  int grid;             // FITRIG_GRID           fused path: CTAs
  int evict_first;      // FITRIG_EVICT_FIRST    fused path: L2 evict_first hint on the streaming loads
  int force_generic;    // FITRIG_FORCE_GENERIC  always take the generic kernel
  int no_pitched_copy;  // FITRIG_NO_PITCHED_COPY fitrig_stream: one copy per snapshot instead of one pitched copy per strip
  int no_pdl;           // FITRIG_NO_PDL         plain launches instead of programmatic dependent launches
  int old_generic;      // FITRIG_OLD_GENERIC    generic path: the three-reads-per-pixel kernel instead of the time-marching one
  int march_cons;       // FITRIG_MARCH_CONS     generic time-marching kernel: consumer warps per CTA
  int march_prod;       // FITRIG_MARCH_PROD     generic time-marching kernel, cp.async variant: producer warps per CTA
  int march_box_kb;     // FITRIG_MARCH_BOX_KB   generic time-marching kernel: target size of a box in KB
  int no_unaligned_fused;  // FITRIG_NO_UNALIGNED_FUSED  unaligned rows: the generic kernel instead of the fused kernel's super-row variant
  int fail_unaligned_encode;  // FITRIG_TEST_FAIL_UNALIGNED_ENCODE  behave as if the driver refused the super-row tensor map (tests the fallback)
};
Tuning read_tuning_env();

// What the tLISI kernels reduce (square cells) and how windows are made of cells (see kernels.cuh, merge_cells_kernel):
// cell == tile and m == 1 in the plain case.
struct CellGeom {
  int cell;  // cell edge in pixels
  int m;     // a window is m x m cells
  int step;  // cells between consecutive windows
};
CellGeom cell_geom(int tile, int stride);
int n_windows(int n, int tile, int stride);  // windows along an axis of n pixels

// Validates and applies defaults.  Returns FITRIG_OK or FITRIG_ERR_INVALID_ARG (+ message in *why).
int normalize_params(int32_t H, int32_t W, int32_t L, const fitrig_params* p, NormParams* out, const char** why);

// Chooses path, tiles per box (consumer warps per CTA), ring depth and grid for `tile_rows` x Tx tiles of U units.
// `rows`: image rows covered by the launch (the whole image, or one strip).
void plan_launch(int tile, int W, int rows, int U, int num_sms, const Tuning& tn, fitrig_plan* plan);
// The fused path's box width, ring depth and grid whatever W % 4 is (the caller has checked that the fused kernel can run);
// extra_row_bytes: what a box row is wider than its tiles (16 for the unaligned variant, kernels.cuh UNAL).
void plan_launch_fused(int tile, int W, int rows, int U, int num_sms, const Tuning& tn, int extra_row_bytes, fitrig_plan* plan);
// Generic time-marching kernel (kernels.cuh, tlisi_march_kernel): boxes of nty x ntx whole cells of c pixels.
constexpr int kMarchMaxCell = 112;     // the ring needs >= 4 boxes of c x c floats in shared memory
constexpr int kMarchMaxWarps = 24;     // warps per CTA (768 threads: up to 85 registers each)
constexpr int kMarchWarps = 23;        // consumer warps of the TMA variant (+ 1 producer warp, one lane of which issues the boxes): the
                                       // inner loop is a chain of dependent shared-memory loads and fp32 operations, so it wants many warps
constexpr int kMarchWarpsCp = 16;      // consumer warps of the cp.async variant ...
constexpr int kMarchProducers = 8;     // ... and its producer warps (16-byte copies: 512 bytes per warp instruction)
constexpr int kMarchTinyCell = 10;     // cells up to this size: one lane per cell (see the kernel)
struct MarchPlan {
  bool ok;        // false: the cell is too large for the ring (the caller takes the three-reads-per-pixel kernel)
  int ntx, nty;   // cells per box
  int bwp, bh;    // box width (floats, multiple of 4, <= 256) and height (<= 256)
  int pitch;      // floats between box rows in shared memory: bwp, or bwp + 8 for the shifted rows of the cp.async variant
  int ngx, ngy;   // boxes per row of boxes, rows of boxes
  int nstage, grid, smem_bytes;
  int ncons, nprod; // consumer and producer warps per CTA
  bool x_aligned; // every box starts on a 16-byte boundary of its row (a condition for fetching it by TMA)
};
MarchPlan plan_march(int c, int W, int rows, int U, int num_sms, const Tuning& tn, bool shifted_rows);
bool fused_tile(int tile);  // N_T the fused kernel serves: 1, 2, 4, 8, 16 (tiles inside a block), 32, and 32 * m (merged blocks)


}  // namespace fitrig
