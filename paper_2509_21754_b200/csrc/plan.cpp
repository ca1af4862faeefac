// plan.cpp -- host-only launch planning (tile grid, time chunking, CTA shape, strip schedule).
#include "plan.h"

#include <stdlib.h>
#include <string.h>

#include <algorithm>

namespace fitrig {

int env_int(const char* name, int dflt) {
  const char* v = getenv(name);
  if (!v || !*v) return dflt;
  return atoi(v);
}

int normalize_params(int32_t H, int32_t W, int32_t L, const fitrig_params* p, NormParams* out, const char** why) {
  fitrig_params z;
  memset(&z, 0, sizeof(z));
  if (!p) p = &z;
  *why = "";
  if (H < 1 || W < 1) { *why = "H and W must be >= 1"; return FITRIG_ERR_INVALID_ARG; }
  if (L < 3) { *why = "need at least 3 snapshots (s = 1..L-2, PAPER.md:155)"; return FITRIG_ERR_INVALID_ARG; }
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
  return FITRIG_OK;
}

// Fused path cost model.  Work items are (tile, time chunk); a warp marches one item through its
// ceil(U/K)+2 snapshots.  One persistent CTA per SM with w warps gives num_sms*w slots, and the
// kernel is bandwidth bound, so a round of items costs ~ w * steps (bytes the slots could have
// moved, busy or idle).  Minimising rounds*steps*w favours (K, w) whose slot count divides the item
// count: e.g. 4096 tiles on 148 SMs -> w = 14 (2 x 2072 slots) instead of 16 (1.73 rounds).
void plan_launch(int tile, int W, int tile_rows, int Tx, int U, int num_sms, fitrig_plan* plan) {
  if (num_sms <= 0) num_sms = 148;
  const bool force_generic = env_int("FITRIG_FORCE_GENERIC", 0) != 0;
  if (tile != kFastTile || (W % 4) != 0 || force_generic) {
    plan->path = 1;
    plan->time_chunks = 1;
    plan->units_per_chunk = U;
    plan->warps_per_cta = 8;
    plan->stages = 0;
    plan->smem_bytes = 0;
    plan->grid = 0;  // sized per launch
    return;
  }
  plan->path = 0;
  const long long tiles = (long long)tile_rows * Tx;
  double best = 1e300;
  int bK = 1, bw = kMaxWarpsPerCta, bs = 3;
  const int maxK = std::min(U, 16);
  for (int K = 1; K <= maxK; ++K) {
    const int cu = (U + K - 1) / K;
    const int Keff = (U + cu - 1) / cu;
    if (Keff != K) continue;
    const int steps = cu + 2;
    for (int w = kMinWarpsPerCta; w <= kMaxWarpsPerCta; ++w) {
      const long long slots = (long long)num_sms * w;
      const long long items = tiles * K;
      const long long rounds = (items + slots - 1) / slots;
      // an SM needs ~6 warps of loads in flight to pull its share of HBM bandwidth; below that a
      // round is latency bound and costs the same as with 6 (so under-filled GPUs prefer more chunks)
      const double per_sm = (double)items / num_sms;
      const double w_eff = std::max(6.0, std::min((double)w, per_sm));
      // small penalties: each extra chunk re-reads 2 halo snapshots; prefer more warps on ties
      double cost = (double)rounds * steps * w_eff * (1.0 + 1e-4 * K) + 1e-3 * (kMaxWarpsPerCta - w);
      if (cost < best) { best = cost; bK = K; bw = w; }
    }
  }
  const int fw = env_int("FITRIG_WARPS", 0), fk = env_int("FITRIG_CHUNKS", 0), fs = env_int("FITRIG_STAGES", 0);
  if (fk > 0) bK = std::min(fk, U);
  if (fw > 0) bw = std::max(1, std::min(fw, kMaxWarpsPerCta));
  const int cu = (U + bK - 1) / bK;
  bK = (U + cu - 1) / cu;
  // deepest ring that fits: stages * warps * 4 KB (+ barriers) <= 227 KB, capped at 4
  bs = std::min(4, (kMaxSmemPerCta - 1024) / (bw * kTileBytes));
  if (fs > 0) bs = std::min(fs, (kMaxSmemPerCta - 1024) / (bw * kTileBytes));
  bs = std::max(2, bs);
  plan->time_chunks = bK;
  plan->units_per_chunk = cu;
  plan->warps_per_cta = bw;
  plan->stages = bs;
  plan->smem_bytes = bw * bs * kTileBytes + bw * bs * 8;
  const long long items = tiles * bK;
  plan->grid = (int)std::min<long long>(num_sms, (items + bw - 1) / bw);
  if (plan->grid < 1) plan->grid = 1;
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
  out->units = L - 2;
  out->Ty = (H + tile - 1) / tile;
  out->Tx = (W + tile - 1) / tile;
  // strip schedule for fitrig_stream: ~256 MiB of snapshot rows per strip (all L snapshots), a multiple of tile
  long long rows = np.strip_rows;
  if (rows == 0) {
    const long long target = 256ll << 20;
    rows = target / ((long long)L * W * 4);
    rows = std::max<long long>(tile, rows / tile * tile);
  }
  const long long Hpad = (long long)out->Ty * tile;
  rows = std::min(rows, Hpad);
  out->strip_rows = (int32_t)rows;
  out->n_strips = (int32_t)((H + rows - 1) / rows);
  out->n_strip_buffers = out->n_strips >= 3 ? 3 : out->n_strips;
  out->strip_buffer_bytes = (int64_t)L * rows * W * 4;
  plan_launch(tile, W, out->Ty, out->Tx, out->units, num_sms, out);
  const int64_t n = (int64_t)out->units * out->Ty * out->Tx;
  out->workspace_bytes = n * (16 + 4 + 4) + (int64_t)out->Ty * out->Tx * 8 + (1 << 20);
  return FITRIG_OK;
}
