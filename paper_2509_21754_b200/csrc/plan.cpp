// plan.cpp -- host-only launch planning (tile grid, time chunking, CTA shape, strip schedule).
#include "plan.h"

#include <stdlib.h>
#include <string.h>

#include <algorithm>
#include <numeric>

namespace fitrig {

static int env_int(const char* name, int dflt) {
  const char* v = getenv(name);
  if (!v || !*v) return dflt;
  return atoi(v);
}

Tuning read_tuning_env() {
  Tuning t;
  t.box_tiles = env_int("FITRIG_BOX_TILES", 0);
  t.stages = env_int("FITRIG_STAGES", 0);
  t.grid = env_int("FITRIG_GRID", 0);
  t.evict_first = env_int("FITRIG_EVICT_FIRST", 0);
  t.force_generic = env_int("FITRIG_FORCE_GENERIC", 0);
  t.no_pitched_copy = env_int("FITRIG_NO_PITCHED_COPY", 0);
  t.no_pdl = env_int("FITRIG_NO_PDL", 0);
  t.old_generic = env_int("FITRIG_OLD_GENERIC", 0);
  t.march_cons = env_int("FITRIG_MARCH_CONS", 0);
  t.march_prod = env_int("FITRIG_MARCH_PROD", 0);
  t.march_box_kb = env_int("FITRIG_MARCH_BOX_KB", 0);
  t.no_unaligned_fused = env_int("FITRIG_NO_UNALIGNED_FUSED", 0);
  t.fail_unaligned_encode = env_int("FITRIG_TEST_FAIL_UNALIGNED_ENCODE", 0);
  return t;
}

int normalize_params(int32_t H, int32_t W, int32_t L, const fitrig_params* p, NormParams* out, const char** why) {
  fitrig_params z;
  memset(&z, 0, sizeof(z));
  if (!p) p = &z;
  *why = "";
  if (H < 1 || W < 1) { *why = "H and W must be >= 1"; return FITRIG_ERR_INVALID_ARG; }
  if (p->accumulate < 0) { *why = "accumulate must be >= 1 (0 selects 1)"; return FITRIG_ERR_INVALID_ARG; }
  out->accumulate = p->accumulate == 0 ? 1 : p->accumulate;
  if (L / out->accumulate < 3) {
    *why = "need at least 3 (accumulated) snapshots (s = 1..L-2, PAPER.md:155)";
    return FITRIG_ERR_INVALID_ARG;
  }
  if (p->tile < 0) { *why = "tile must be >= 1 (0 selects the default 32)"; return FITRIG_ERR_INVALID_ARG; }
  if (p->ref_mode < 0 || p->ref_mode > 2) { *why = "unknown ref_mode"; return FITRIG_ERR_INVALID_ARG; }
  if (p->branch < 0 || p->branch > 1) { *why = "unknown branch"; return FITRIG_ERR_INVALID_ARG; }
  if (p->device < 0) { *why = "device ordinal must be >= 0"; return FITRIG_ERR_INVALID_ARG; }
  if (p->C > 0.f && p->C < 1e-30f) { *why = "C must be >= 1e-30 (or <= 0 for the default 1e-6)"; return FITRIG_ERR_INVALID_ARG; }
  if (!(p->M_override >= 0.f)) { *why = "M_override must be >= 0"; return FITRIG_ERR_INVALID_ARG; }
  out->tile = p->tile == 0 ? kFastTile : p->tile;
  out->C = p->C > 0.f ? p->C : 1e-6f;
  out->ref_mode = p->ref_mode;
  out->M_override = p->M_override;
  out->branch = p->branch;
  out->device = p->device;
  if (p->strip_rows < 0 || (p->strip_rows % out->tile) != 0) {
    *why = "strip_rows must be a non-negative multiple of tile";
    return FITRIG_ERR_INVALID_ARG;
  }
  out->strip_rows = p->strip_rows;
  out->stride = p->stride == 0 ? out->tile : p->stride;
  if (out->stride < 1 || out->tile % out->stride != 0) {
    *why = "stride must divide tile (0 selects tile: non-overlapping tiles)";
    return FITRIG_ERR_INVALID_ARG;
  }
  if (out->stride != out->tile && (p->branch != 0 || out->accumulate != 1 || p->row_offset != 0)) {
    *why = "overlapping windows (stride < tile): image branch, no accumulation, no row shards";
    return FITRIG_ERR_INVALID_ARG;
  }
  out->harmonics = p->harmonics == 0 ? 1 : p->harmonics;
  if (out->harmonics < 1 || out->harmonics > 32 || (out->harmonics & (out->harmonics - 1)) != 0) {
    *why = "harmonics must be 1, 2, 4, 8, 16 or 32 (0 selects 1)";
    return FITRIG_ERR_INVALID_ARG;
  }
  if (p->row_offset < 0 || (p->row_offset % out->tile) != 0) {
    *why = "row_offset must be a non-negative multiple of tile";
    return FITRIG_ERR_INVALID_ARG;
  }
  out->row_offset = p->row_offset;
  if (p->batch < 0) { *why = "batch must be >= 1 (0 selects 1)"; return FITRIG_ERR_INVALID_ARG; }
  out->batch = p->batch == 0 ? 1 : p->batch;
  if (out->batch > 1 && (p->row_offset != 0 || out->stride != out->tile)) {
    *why = "batch > 1: no row shards, no overlapping windows";
    return FITRIG_ERR_INVALID_ARG;
  }
  const long long U = (long long)L / out->accumulate - 2;
  if (p->branch == FITRIG_BRANCH_FREQUENCY && U > 8192) {
    *why = "frequency branch: at most 8192 units (the twiddle table of the temporal DFT lives in shared memory)";
    return FITRIG_ERR_INVALID_ARG;
  }
  return FITRIG_OK;
}

// Fused path: one persistent CTA per SM; a consumer warp owns a 32x32 pixel block = (32 / N_T)^2 tiles for
// cells of 32, 16 or 8 pixels (a lane holds several tiles for 4, 2, 1), and the CTAs share the G = boxes * U (box column, unit) pairs evenly (see
// kernels.cuh), so only the box width, ring depth and grid are chosen here.  A box of 8 adjacent blocks is
// 32 rows of 1 KB: long enough bursts for HBM to run at its streaming rate.  6 boxes of 32 KB in flight per
// SM are about 3x the HBM latency-bandwidth product (~65 KB per SM).
CellGeom cell_geom(int tile, int stride) {
  CellGeom g;
  if (stride == tile) {
    // non-overlapping: tiles of 32 * m pixels are m x m blocks of 32; a tile with a divisor of 16, 8 or 4 pixels (12, 24,
    // 48, 100 ...) is m x m cells of that size, which the fused kernel reduces at (nearly) the rate of a plain read;
    // everything else (5, 7, 9, 10 ...) is its own cell and takes the generic time-marching kernel
    g.cell = tile; g.m = 1; g.step = 1;
    if (!fused_tile(tile)) {
      bool found = false;
      for (int d = 16; d >= 4 && !found; d >>= 1)
        if (tile % d == 0) { g.cell = d; g.m = tile / d; g.step = g.m; found = true; }
      // no such divisor and more than 32 pixels (50, 66, 98 ...): the generic kernel is at its best on cells of at most
      // 32 pixels (a warp takes whole cell rows), so the largest divisor in 5 .. 32 becomes the cell
      for (int d = 32; d >= 5 && !found && tile > kFastTile; --d)
        if (tile % d == 0) { g.cell = d; g.m = tile / d; g.step = g.m; found = true; }
    } else if (tile > kFastTile) {
      g.cell = kFastTile; g.m = tile / kFastTile; g.step = g.m;
    }
  } else if (stride % kFastTile == 0) {
    g.cell = kFastTile; g.m = tile / kFastTile; g.step = stride / kFastTile;
  } else {
    g.cell = stride; g.m = tile / stride; g.step = 1;
  }
  return g;
}

int n_windows(int n, int tile, int stride) {
  if (stride == tile) return (n + tile - 1) / tile;  // R5: a partial last tile
  const int cells = (n + stride - 1) / stride, m = tile / stride;
  return std::max(1, cells - m + 1);  // R27
}

bool fused_tile(int tile) {
  return tile == 16 || tile == 8 || tile == 4 || tile == 2 || tile == 1 || (tile >= kFastTile && tile % kFastTile == 0);
}

void plan_launch(int tile, int W, int rows, int U, int num_sms, const Tuning& tn, fitrig_plan* plan) {
  const bool force_generic = tn.force_generic != 0;
  if (!fused_tile(tile) || (W % 4) != 0 || force_generic) {
    plan->path = 1;
    plan->units_per_cta = 0;
    plan->box_tiles = 0;
    plan->warps_per_cta = 8;
    plan->stages = 0;
    plan->smem_bytes = 0;
    plan->grid = 0;  // sized per launch
    return;
  }
  plan_launch_fused(tile, W, rows, U, num_sms, tn, 0, plan);
}

void plan_launch_fused(int tile, int W, int rows, int U, int num_sms, const Tuning& tn, int extra_row_bytes, fitrig_plan* plan) {
  if (num_sms <= 0) num_sms = 148;
  plan->path = 0;
  const int rows32 = (rows + kFastTile - 1) / kFastTile, Tx32 = (W + kFastTile - 1) / kFastTile;
  const int fb = tn.box_tiles, fs = tn.stages, fg = tn.grid;
  // (a TMA box is at most 256 elements wide: the unaligned variant's boxes are 4 floats wider than their tiles)
  int ntw = std::min(extra_row_bytes ? kMaxTilesPerBox - 1 : kMaxTilesPerBox, Tx32);
  auto pairs = [&](int n) { return (long long)rows32 * ((Tx32 + n - 1) / n) * U; };
  // small problems are latency bound: narrower boxes give more CTAs something to do
  while (ntw > 1 && (pairs(ntw) + kMinUnitsPerCta - 1) / kMinUnitsPerCta < num_sms) ntw = (ntw + 1) / 2;
  if (fb > 0) ntw = std::max(1, std::min(fb, std::min(extra_row_bytes ? kMaxTilesPerBox - 1 : kMaxTilesPerBox, Tx32)));
  const long long G = pairs(ntw);
  int grid = (int)std::max<long long>(1, std::min<long long>(num_sms, (G + kMinUnitsPerCta - 1) / kMinUnitsPerCta));
  if (fg > 0) grid = fg;
  const int per_edge = (tile < kFastTile && tile >= 8) ? kFastTile / tile : 1;
  const int groups = per_edge * per_edge;  // tiles per warp that keep an arg-max scratch (tiles below 8 pixels need none)
  const int scratch = ntw * groups * kScratchVec * 16;
  const int box_bytes = ntw * kTileBytes + kFastTile * extra_row_bytes;
  const int fit = (kMaxSmemPerCta - 2048 - scratch) / box_bytes;
  int stages = std::min(6, fit);
  if (fs > 0) stages = std::min(fs, fit);
  stages = std::max(2, std::min(stages, kMaxStages));
  plan->box_tiles = ntw;
  plan->warps_per_cta = ntw + 1;  // consumers + the producer
  plan->stages = stages;
  plan->grid = grid;
  plan->units_per_cta = (int32_t)((G + grid - 1) / grid);
  plan->smem_bytes = stages * box_bytes + 2 * kMaxStages * 8 + scratch;  // ring, mbarriers, scratch
}

MarchPlan plan_march(int c, int W, int rows, int U, int num_sms, const Tuning& tn, bool shifted_rows) {
  MarchPlan m;
  memset(&m, 0, sizeof(m));
  if (num_sms <= 0) num_sms = 148;
  if (c < 1 || c > kMarchMaxCell || U < 1) return m;
  const int cells_x = (W + c - 1) / c, cells_y = (rows + c - 1) / c;
  auto width = [&](int ntx) { return (ntx * c + 3) / 4 * 4; };
  // cp.async variant: a box is shifted by up to 3 floats, the last 16-byte copy of a row may overhang by 3 more, and the
  // pitch must be congruent to W modulo 4 (global and shared addresses then agree modulo 16 bytes in every row)
  auto pad_of = [&](int bw) { return shifted_rows ? 8 + (((W - bw - 8) % 4) + 4) % 4 : 0; };
  const int pad = shifted_rows ? 11 : 0;  // (the largest pad_of: sizes the boxes)
  int ntx = std::max(1, std::min(cells_x, 256 / c));
  if (c <= kMarchTinyCell && ntx > 32) ntx = 32;  // cells of a few pixels: a warp takes 32 adjacent cells, one per lane
  while (ntx > 1 && (width(ntx) > 256 || (long long)(width(ntx) + pad) * c * 4 > 48 * 1024)) --ntx;  // >= 4 boxes in the ring
  // boxes of about 32 KB (the fused kernel's box): long rows for HBM, several boxes in flight per SM
  int nprod = shifted_rows ? kMarchProducers : 1;
  if (shifted_rows && tn.march_prod > 0) nprod = std::min(tn.march_prod, kMarchMaxWarps - 1);
  int kWarps = shifted_rows ? kMarchWarpsCp : kMarchWarps;  // consumer warps of the kernel
  if (tn.march_cons > 0) kWarps = tn.march_cons;
  kWarps = std::max(1, std::min(kWarps, kMarchMaxWarps - nprod));
  const int box_target = (tn.march_box_kb > 0 ? tn.march_box_kb : 32) * 1024;
  auto rows_fit = [&](int bytes) { return std::max(1, std::min(std::min(cells_y, 256 / c), bytes / ((width(ntx) + pad) * 4 * c))); };
  int nty = rows_fit(box_target);
  auto pairs = [&](int nx, int ny) { return (long long)((cells_x + nx - 1) / nx) * ((cells_y + ny - 1) / ny) * U; };
  // small problems are latency bound: smaller boxes give more CTAs something to do
  bool shrunk = false;
  while ((pairs(ntx, nty) + kMinUnitsPerCta - 1) / kMinUnitsPerCta < num_sms && (nty > 1 || ntx > 1)) {
    if (nty > 1) nty = (nty + 1) / 2;
    else ntx = (ntx + 1) / 2;
    shrunk = true;
  }
  if (!shrunk) {
    // the consumer warps share a box's items (a row of floor(32 / c) adjacent cells, or one cell when c > 32): prefer
    // the box height, up to 40 KB, that leaves the fewest warps idle in the last round
    const int per_row = (c <= kMarchTinyCell) ? (ntx + 31) / 32 : (c <= 32) ? (ntx + 32 / c - 1) / (32 / c) : ntx;
    auto eff = [&](int ny) { const int it = ny * per_row; return (double)it / (double)((it + kWarps - 1) / kWarps * kWarps); };
    int best = nty;
    for (int ny = std::max(1, nty / 2); ny <= rows_fit(box_target + box_target / 4); ++ny)
      if (eff(ny) > eff(best) + 1e-9 || (eff(ny) > eff(best) - 1e-9 && ny > best && ny <= nty)) best = ny;
    nty = best;
  }
  // box columns start at multiples of ntx * c pixels: keep them on 16-byte boundaries where the cell size allows
  // (TMA faults on other box origins; where it cannot be had the kernel copies with cp.async instead, see x_aligned)
  const int qx = 4 / std::gcd(c, 4);
  if (ntx < cells_x && ntx >= qx) ntx = ntx / qx * qx;
  m.x_aligned = (ntx >= cells_x) || ((ntx * c) % 4 == 0);
  m.ncons = kWarps; m.nprod = nprod;
  m.ntx = ntx; m.nty = nty; m.bwp = width(ntx); m.bh = nty * c; m.pitch = m.bwp + pad_of(m.bwp);
  m.ngx = (cells_x + ntx - 1) / ntx; m.ngy = (cells_y + nty - 1) / nty;
  const int slot = (m.bh * m.pitch * 4 + 127) / 128 * 128;
  int stages = std::min(kMaxStages, (kMaxSmemPerCta - 2048) / slot);
  if (tn.stages > 0) stages = std::min(stages, std::max(4, tn.stages));
  if (stages < 4) return m;  // three snapshots in use + one in flight
  m.nstage = stages;
  const long long G = pairs(ntx, nty);
  m.grid = (int)std::max<long long>(1, std::min<long long>(num_sms, (G + kMinUnitsPerCta - 1) / kMinUnitsPerCta));
  if (tn.grid > 0) m.grid = tn.grid;
  m.smem_bytes = stages * slot + 2 * kMaxStages * 8;
  m.ok = G <= 0x7fffffffll;
  return m;
}

}  // namespace fitrig

using namespace fitrig;

extern "C" int fitrig_plan_query(int32_t H, int32_t W, int32_t L, const fitrig_params* params, int32_t num_sms,
                                 fitrig_plan* out) {
  if (!out) return FITRIG_ERR_INVALID_ARG;
  NormParams np;
  const char* why = "";
  int rc = normalize_params(H, W, L, params, &np, &why);
  if (rc != FITRIG_OK) return rc;
  memset(out, 0, sizeof(*out));
  const int tile = np.tile;
  out->units = L / np.accumulate - 2;
  out->Ty = n_windows(H, tile, np.stride);
  out->Tx = n_windows(W, tile, np.stride);
  const int cell = cell_geom(tile, np.stride).cell;
  // strip schedule for fitrig_stream: ~256 MiB of snapshot rows per strip (all L snapshots), a multiple of tile
  long long rows = np.strip_rows;
  if (rows == 0) {
    const long long target = 256ll << 20;
    rows = target / ((long long)L * W * 4);
    // whole tiles, and whole 32-row blocks when the cells ride the fused path
    const long long q = (kFastTile % cell == 0) ? std::lcm((long long)tile, (long long)kFastTile) : tile;
    rows = std::max<long long>(q, rows / q * q);
  }
  const long long Hpad = ((long long)H + tile - 1) / tile * tile;
  rows = std::min(rows, Hpad);
  out->strip_rows = (int32_t)rows;
  out->n_strips = (int32_t)((H + rows - 1) / rows);
  out->n_strip_buffers = out->n_strips >= 3 ? 3 : out->n_strips;
  out->strip_buffer_bytes = (int64_t)L * rows * W * 4;
  const Tuning tn = read_tuning_env();
  plan_launch(cell, W, H, out->units, num_sms, tn, out);
  if (out->path == 1 && W % 4 != 0 && cell <= kFastTile && fused_tile(cell) && np.accumulate == 1 && !tn.force_generic &&
      !tn.no_unaligned_fused && ((long long)L * H) % (4 / std::gcd(W, 4)) == 0)
    plan_launch_fused(cell, W, H, out->units, num_sms, tn, 16, out);  // the super-row variant (kernels.cuh, UNAL)
  const int64_t n = (int64_t)np.batch * out->units * out->Ty * out->Tx;
  out->workspace_bytes = n * (16 + 4 + 4) + (int64_t)out->Ty * out->Tx * 8 + (1 << 20);
  return FITRIG_OK;
}
