// kernels.cuh -- sm_100a CUDA kernels of the FITrig hot path (arxiv 2509.21754).
//
//   tlisi_fused_kernel    steps a1-a5: |x_{s+1}-x_s|, second difference, clamped ratio, per-tile
//                         sum/max/argmax/sum and the global maximum, in ONE pass that reads every
//                         snapshot byte once.  A warp owns one 32x32 tile and marches it through
//                         time; a producer warp fetches rows of up to 8 adjacent tiles as single TMA
//                         boxes (cp.async.bulk.tensor) into a CTA-wide ring guarded by full/empty mbarriers.
//   tlisi_generic_kernel  the same per-tile quantities for any tile size / alignment (3 reads per pixel-unit).
//   stack_max_kernel      global maximum for the generic path.
//   finalize_kernel       step a6-a7: q = mean(D)*max(D)*mean(r)/M^2, tLISI = 1-q, per-unit mean/std.
//   spectrum_kernel       step a10: per-tile temporal DFT, eta = max |F_k|, k*.
//   compact_kernel        step a8: z-score, strict threshold, ordered compaction (ballot + prefix sums).
//
// Citations: PAPER.md line numbers; R<n> = readings in DESIGN.md.
#pragma once
#include <cuda.h>
#include <cuda_runtime.h>
#include <stdint.h>

#include "fitrig.h"
#include "plan.h"

namespace fitrig {

// Per-tile, per-unit partial results of Eq. 6: sum Delta, max Delta, sum r, and the
// tile-relative position (row * N_T + col) of the first max-Delta pixel (R20).  16 bytes.
struct __align__(16) RawTile {
  float sumD;
  float maxD;
  float sumR;
  int32_t pos;
};

// Cells of ONE pixel ("per-pixel detection"; overlapping windows at stride 1): sum Delta = max Delta =
// Delta and the position is 0, so the record shrinks to {Delta, r}: 8 bytes instead of 16 (the per-pixel map of a
// 64 x 2048 x 2048 stack is 260 M records: 2 GB less to write and 2 GB less to read back).  Such a context keeps its
// cell records in this form in the same buffer (`pix8` in the kernel parameters).
struct __align__(8) RawPix {
  float delta;
  float r;
};
__device__ __forceinline__ RawTile load_raw(const RawTile* raw, long long i, int pix8) {
  if (!pix8) return raw[i];
  const RawPix v = reinterpret_cast<const RawPix*>(raw)[i];
  RawTile o; o.sumD = v.delta; o.maxD = v.delta; o.sumR = v.r; o.pos = 0;
  return o;
}
__device__ __forceinline__ void store_raw(RawTile* raw, long long i, int pix8, float S, float Mx, float R, int pos) {
  if (pix8) {
    RawPix v; v.delta = Mx; v.r = R;
    reinterpret_cast<RawPix*>(raw)[i] = v;
  } else {
    RawTile o; o.sumD = S; o.maxD = Mx; o.sumR = R; o.pos = pos;
    raw[i] = o;
  }
}

// ---------------------------------------------------------------------------------------------
// small device helpers
// ---------------------------------------------------------------------------------------------
__device__ __forceinline__ uint32_t smem_u32(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }

__device__ __forceinline__ void mbar_init(uint32_t bar, uint32_t count) {
  asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(bar), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_arrive_expect_tx(uint32_t bar, uint32_t bytes) {
  asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(bar), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_arrive(uint32_t bar) {
  asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(bar) : "memory");
}
__device__ __forceinline__ void mbar_wait(uint32_t bar, uint32_t parity) {
  uint32_t done;
  do {
    asm volatile(
        "{\n\t.reg .pred p;\n\t"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n\t"
        "selp.u32 %0, 1, 0, p;\n\t}"
        : "=r"(done)
        : "r"(bar), "r"(parity)
        : "memory");
  } while (!done);
}
__device__ __forceinline__ uint64_t l2_evict_first_policy() {
  uint64_t pol;
  asm volatile("createpolicy.fractional.L2::evict_first.b64 %0, 1.0;" : "=l"(pol));
  return pol;
}
// One box (ntw * 32 columns x 32 rows, fp32) of snapshot z at pixel (x, y) -> shared memory; completes on `bar`.
__device__ __forceinline__ void tma_load_box_hint(uint32_t dst, const CUtensorMap* map, uint32_t bar, int x, int y, int z,
                                                  uint64_t policy) {
  asm volatile(
      "cp.async.bulk.tensor.3d.shared::cluster.global.mbarrier::complete_tx::bytes.L2::cache_hint"
      " [%0], [%1, {%2, %3, %4}], [%5], %6;" ::"r"(dst),
      "l"(map), "r"(x), "r"(y), "r"(z), "r"(bar), "l"(policy)
      : "memory");
}
__device__ __forceinline__ void tma_load_box(uint32_t dst, const CUtensorMap* map, uint32_t bar, int x, int y, int z) {
  asm volatile(
      "cp.async.bulk.tensor.3d.shared::cluster.global.mbarrier::complete_tx::bytes"
      " [%0], [%1, {%2, %3, %4}], [%5];" ::"r"(dst),
      "l"(map), "r"(x), "r"(y), "r"(z), "r"(bar)
      : "memory");
}
__device__ __forceinline__ void tma_load_box2d(uint32_t dst, const CUtensorMap* map, uint32_t bar, int x, int y) {
  asm volatile(
      "cp.async.bulk.tensor.2d.shared::cluster.global.mbarrier::complete_tx::bytes"
      " [%0], [%1, {%2, %3}], [%4];" ::"r"(dst),
      "l"(map), "r"(x), "r"(y), "r"(bar)
      : "memory");
}
// Programmatic dependent launch: a kernel launched with cudaLaunchAttributeProgrammaticStreamSerialization may become
// resident while its predecessor in the stream still runs; pdl_wait() blocks until the predecessor has completed and
// its memory is visible (a no-op for a plain launch).  pdl_launch_dependents() lets the successor's CTAs be scheduled.
__device__ __forceinline__ void pdl_wait() { asm volatile("griddepcontrol.wait;" ::: "memory"); }
__device__ __forceinline__ void pdl_launch_dependents() { asm volatile("griddepcontrol.launch_dependents;" ::: "memory"); }
__device__ __forceinline__ float rcp_approx(float a) {
  float r;
  asm("rcp.approx.ftz.f32 %0, %1;" : "=f"(r) : "f"(a));
  return r;
}
// order-preserving float -> uint key (so atomicMax / redux.max on uints orders signed floats)
__device__ __forceinline__ unsigned float_to_key(float f) {
  unsigned b = __float_as_uint(f);
  return (b & 0x80000000u) ? ~b : (b | 0x80000000u);
}
__host__ __device__ __forceinline__ float key_to_float(unsigned k) {
  unsigned b = (k & 0x80000000u) ? (k & 0x7fffffffu) : ~k;
#ifdef __CUDA_ARCH__
  return __uint_as_float(b);
#else
  float f;
  memcpy(&f, &b, 4);
  return f;
#endif
}

// Clamped ratio r of Eq. 4-5 for one pixel: delta >= 0, ref = x^(s+1).
//   ABS     x_hat = |ref|, |ref| == 0 -> C     r = min(delta / x_hat, 1)
//   LITERAL x_hat = ref,   ref == 0   -> C     (r may be negative)
//   FLOOR   x_hat = max(ref, C)
// delta * rcp saturates to [0,1]; the saturating multiply also maps 0 * inf (= NaN) to 0, which is
// the value Eq. 5 gives (R8).
template <int REF_MODE>
__device__ __forceinline__ float clamped_ratio(float delta, float ref, float C) {
  if (REF_MODE == FITRIG_REF_ABS) {
    float a = fabsf(ref);
    a = (a == 0.f) ? C : a;
    return __saturatef(delta * rcp_approx(a));
  } else if (REF_MODE == FITRIG_REF_LITERAL) {
    float a = (ref == 0.f) ? C : ref;
    float qv = delta * rcp_approx(a);
    qv = (qv != qv) ? 0.f : qv;  // 0 * inf
    return fminf(qv, 1.f);
  } else {
    float a = fmaxf(ref, C);
    return __saturatef(delta * rcp_approx(a));
  }
}

// ---------------------------------------------------------------------------------------------
// Fused time-marching tLISI kernel (N_T = 32)
// ---------------------------------------------------------------------------------------------
struct FusedParams {
  RawTile* raw;          // [U][Ty][Tx] whole map
  unsigned* gmax_key;    // ordered key of the running global maximum (atomicMax)
  const float* base;     // snapshot 0 of this launch's rows (the memory the TMA descriptor covers)
  long long snap_stride; // elements between consecutive snapshots
  int W;                 // image width (row pitch in elements)
  int Tx, Ty;            // grid of the cells this launch reduces, over the whole map (cells of 1 .. 32 pixels)
  int Tx32;              // 32-pixel block columns = ceil(W / 32): a consumer warp owns one 32x32 block
  int rows_tiles;        // rows of 32x32 blocks covered by this launch (whole image, or one strip)
  int ty_base;           // first tile row (in tiles of N_T) of this launch inside the whole map
  int ty_end;            // one past the last cell row this launch owns: min(Ty, ty_base + ceil(rows / cell)).  A strip whose
                         // height is not a multiple of 32 shares its last 32-row block with the next strip; the cells of
                         // the zero-filled overhang belong to that strip and are neither written nor re-read here
  int U;                 // units = L - 2
  int ntw;               // tiles per TMA box = consumer warps per CTA (1..kMaxTilesPerBox)
  int ngx;               // boxes per tile row = ceil(Tx / ntw)
  int nstage;            // depth of the CTA's ring of boxes
  int G;                 // rows_tiles * ngx * U: (box column, unit) pairs of this launch, box-major
  int evict_first;       // L2 policy of the streaming loads
  int z0, zmask;         // snapshot s of the launch lives in slot (z0 + s) & zmask: real-time ring of 4 slots: zmask = 3;
                         // a plain stack: z0 = 0, zmask = 0x7fffffff (no modulo, no branch in the lane-0 paths)
  int acc;               // snapshot accumulation: image j of the method = sum of raw snapshots g*j .. g*j+g-1
  int k_rows, a_off, rows;  // the unaligned variant (UNAL): image rows per super row, floats between the 16-byte boundary
                            // below the base pointer and the base, image rows per snapshot of this launch
  int srows;                // UNAL: rows between consecutive snapshots (snap_stride / W; >= rows: the last strip is shorter)
  int even_shifts;          // UNAL: every row starts on an 8-byte boundary (W and a_off even)
  int dep;               // programmatic dependent launch (see pdl_wait): 1 = this grid must not touch memory before the grid
                         // ahead of it in the stream has completed (wait at the start, after the prologue); 2 = the grid
                         // ahead is an independent tLISI launch of the same call (another stack of a batch): run beside
                         // its tail, but do not COMPLETE before it has (wait at the end), so that the finalise kernel,
                         // which waits for the last of the chain, finds all of them done; 0 = a plain launch
  float C;
};

__device__ __forceinline__ int ring_slot(int z0, int zmask, int s) { return (z0 + s) & zmask; }

// Work distribution: a "group" is a row of ntw horizontally adjacent tiles, fetched as ONE TMA box of
// 32 rows x (ntw * 128) contiguous bytes (isolated 128-byte rows cost ~15 % of the HBM bandwidth, see
// profiles/).  The G (group, unit) pairs of a launch, ordered group-major / time-minor, are cut into
// one contiguous range per CTA (range c = [c*G/n, (c+1)*G/n)), so every CTA carries the same load
// whatever the tile count.  A range is walked as "segments": a run of consecutive units of one
// group, which costs its units + 2 snapshots to march through (the 2-snapshot halo is re-read only
// where a cut falls inside a group's time series: at most once per CTA).
struct Segment {
  int gx, ty_local, u0, nsteps;  // box column, tile row, first unit, snapshots to load (= units + 2)
};

__device__ __forceinline__ Segment decode_segment(const FusedParams& p, int g, int g_end) {
  Segment c;
  const int group = g / p.U;
  c.u0 = g - group * p.U;
  c.ty_local = group / p.ngx;
  c.gx = group - c.ty_local * p.ngx;
  c.nsteps = min(p.U - c.u0, g_end - g) + 2;
  return c;
}

__device__ __forceinline__ void cp_async16(uint32_t dst, const void* src) {
  asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"(dst), "l"(src) : "memory");
}
__device__ __forceinline__ void cp_async4_zfill(uint32_t dst, const void* src, int src_bytes) {
  asm volatile("cp.async.ca.shared.global [%0], [%1], 4, %2;" ::"r"(dst), "l"(src), "r"(src_bytes) : "memory");
}
__device__ __forceinline__ void cp_async8_zfill(uint32_t dst, const void* src, int src_bytes) {
  asm volatile("cp.async.ca.shared.global [%0], [%1], 8, %2;" ::"r"(dst), "l"(src), "r"(src_bytes) : "memory");
}
__device__ __forceinline__ void cp_async_mbar_arrive_noinc(uint32_t bar) {
  asm volatile("cp.async.mbarrier.arrive.noinc.shared::cta.b64 [%0];" ::"r"(bar) : "memory");
}
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;" ::: "memory"); }
__device__ __forceinline__ void cp_async_wait_all() { asm volatile("cp.async.wait_group 0;" ::: "memory"); }

// Which pixels of its warp's 32x32 block a lane holds, for tiles of T = 32, 16 or 8 pixels.  The block is
// (32/T)^2 tiles; T*T/32 lanes share one tile, so that the 32 pixels of a lane belong to ONE tile and every
// reduction is a butterfly over the tile's lane group.  A lane reads float4's: T/4 lanes cover a tile row, the
// group covers T/8 rows per load, 8 loads cover the tile; pixels are held in row-major order of the tile.
// In every geometry a quarter warp (8 consecutive lanes) reads ONE 128-byte row of the block (conflict free):
//   T = 32  lane = [row 2 bits][col 3 bits]                  one tile, all 32 lanes
//   T = 16  lane = [sub_row][row parity][sub_col][col 2 bits]  the two tiles of a block row share the quarter warp:
//           a tile's 8 lanes are NOT consecutive (they differ in bits 0, 1 and 3)
//   T = 8   lane = [sub_row 2 bits][sub_col 2 bits][col 1 bit] a tile's 2 lanes are neighbours
// XOR*: the lane-index bits that vary inside a tile's group (butterfly offsets); SPLIT is the one used first.
template <int T>
struct LaneGeom;
template <>
struct LaneGeom<32> {
  static constexpr int LPT = 32, RPL = 4, NSUB = 1, SPLIT = 16, NREST = 4;
  __device__ static __forceinline__ int rest(int i) { return 8 >> i; }  // 8, 4, 2, 1
  __device__ static __forceinline__ int sub_row(int) { return 0; }
  __device__ static __forceinline__ int sub_col(int) { return 0; }
  __device__ static __forceinline__ int row_in_tile(int lane) { return lane >> 3; }   // + RPL * j
  __device__ static __forceinline__ int col_in_tile(int lane) { return (lane & 7) * 4; }
  __device__ static __forceinline__ int leader_lane(int) { return 0; }
};
template <>
struct LaneGeom<16> {
  static constexpr int LPT = 8, RPL = 2, NSUB = 2, SPLIT = 8, NREST = 2;
  __device__ static __forceinline__ int rest(int i) { return 2 >> i; }  // 2, 1
  __device__ static __forceinline__ int sub_row(int lane) { return lane >> 4; }
  __device__ static __forceinline__ int sub_col(int lane) { return (lane >> 2) & 1; }
  __device__ static __forceinline__ int row_in_tile(int lane) { return (lane >> 3) & 1; }
  __device__ static __forceinline__ int col_in_tile(int lane) { return (lane & 3) * 4; }
  __device__ static __forceinline__ int leader_lane(int lane) { return lane & 0x14; }
};
template <>
struct LaneGeom<8> {
  static constexpr int LPT = 2, RPL = 1, NSUB = 4, SPLIT = 1, NREST = 0;
  __device__ static __forceinline__ int rest(int) { return 0; }
  __device__ static __forceinline__ int sub_row(int lane) { return lane >> 3; }
  __device__ static __forceinline__ int sub_col(int lane) { return (lane >> 1) & 3; }
  __device__ static __forceinline__ int row_in_tile(int) { return 0; }
  __device__ static __forceinline__ int col_in_tile(int lane) { return (lane & 1) * 4; }
  __device__ static __forceinline__ int leader_lane(int lane) { return lane & ~1; }
};
template <int T>
__device__ __forceinline__ int geom_block_row(int lane) { return LaneGeom<T>::sub_row(lane) * T + LaneGeom<T>::row_in_tile(lane); }
template <int T>
__device__ __forceinline__ int geom_block_col(int lane) { return LaneGeom<T>::sub_col(lane) * T + LaneGeom<T>::col_in_tile(lane); }

// Which row of its warp's 32x32 block the j-th float4 (j = 0..7) of a lane comes from; its columns are 4 (lane & 7) ..
// for LT = 32, 4, 2 and geom_block_col<LT> otherwise.  LT = 32, 16, 8: LaneGeom above.  Tiles of 4 and 2 pixels: a lane
// holds WHOLE tiles (no reduction across lanes): lane = [rq 2 bits][cg 3 bits],
//   LT = 4  rows 16 (j / 4) + 4 rq + j % 4: the two 4x4 tiles (tile row rq and rq + 4, tile column cg)
//   LT = 2  rows  8 (j / 2) + 2 rq + j % 2: the eight 2x2 tiles (tile rows rq + 4 (j / 2), tile columns 2 cg, 2 cg + 1)
// In every geometry a quarter warp reads one 128-byte row per load (conflict free).
template <int LT>
__device__ __forceinline__ int lane_row(int lane, int j) {
  if (LT == 4) return 16 * (j >> 2) + 4 * (lane >> 3) + (j & 3);
  if (LT == 2) return 8 * (j >> 1) + 2 * (lane >> 3) + (j & 1);
  return geom_block_row<(LT == 4 || LT == 2) ? 32 : LT>(lane) + LaneGeom<(LT == 4 || LT == 2) ? 32 : LT>::RPL * j;
}
template <int LT>
__device__ __forceinline__ int lane_col(int lane) { return geom_block_col<(LT == 4 || LT == 2) ? 32 : LT>(lane); }

// The lane's 32 pixels out of a box (row pitch `pitch` bytes) into registers / added to registers.
template <int LT>
__device__ __forceinline__ void load_tile(float (&N)[32], const unsigned char* block_ptr, int pitch, int lane) {
  const unsigned char* src = block_ptr + lane_col<LT>(lane) * 4;
#pragma unroll
  for (int j = 0; j < 8; ++j) {
    const float4 t = *reinterpret_cast<const float4*>(src + lane_row<LT>(lane, j) * pitch);
    N[4 * j] = t.x; N[4 * j + 1] = t.y; N[4 * j + 2] = t.z; N[4 * j + 3] = t.w;
  }
}

template <int LT>
__device__ __forceinline__ void add_tile(float (&N)[32], const unsigned char* block_ptr, int pitch, int lane) {
  const unsigned char* src = block_ptr + lane_col<LT>(lane) * 4;
#pragma unroll
  for (int j = 0; j < 8; ++j) {
    const float4 t = *reinterpret_cast<const float4*>(src + lane_row<LT>(lane, j) * pitch);
    N[4 * j] += t.x; N[4 * j + 1] += t.y; N[4 * j + 2] += t.z; N[4 * j + 3] += t.w;
  }
}

// Running signed maximum (a5) and the smallest magnitude of a freshly loaded tile.  zmin == 0 tells
// the NEXT step, whose reference image this tile is, that Eq. 5's "x == 0 -> C" case occurs.
__device__ __forceinline__ void scan_tile(const float (&N)[32], float& gmax, float& zmin) {
  float z = 3.402823466e38f;
#pragma unroll
  for (int k = 0; k < 32; ++k) {
    gmax = fmaxf(gmax, N[k]);
    z = fminf(z, fabsf(N[k]));
  }
  zmin = z;
}

// Steps a1-a4 for the 32 pixels of one lane: N = x^(s+2) (new), X = x^(s+1) (reference image,
// PAPER.md:203), dp = signed x^(s+1) - x^(s).  Returns the lane's sum Delta, sum r, max Delta and the
// index j (0..7) of the first 4-pixel group that attains it; dp becomes x^(s+2) - x^(s+1).
//
// REF_ABS: r = sat(Delta * rcp(|x|)).  rcp(0) = +inf, so a zero reference pixel yields 1 (Delta > 0)
// or sat(NaN) = 0 (Delta == 0) instead of Eq. 5's min(Delta / C, 1); `zero_ref` (warp uniform, known
// from scan_tile one step earlier) adds the difference first, so the per-pixel x == 0 test leaves
// the hot loop.
template <int REF_MODE>
__device__ __forceinline__ void tile_step(const float (&N)[32], const float (&X)[32], float (&dp)[32], float C,
                                          bool zero_ref, float& S, float& R, float& Mx, int& jmax) {
  float S0 = 0.f, S1 = 0.f, R0 = 0.f, R1 = 0.f;
  Mx = 0.f;
  jmax = 0;
  if (REF_MODE == FITRIG_REF_ABS && zero_ref) {
    const float invC = rcp_approx(C);
#pragma unroll
    for (int k = 0; k < 32; ++k) {
      if (X[k] == 0.f) {
        const float delta = fabsf(fabsf(N[k] - X[k]) - fabsf(dp[k]));
        R0 += __saturatef(delta * invC) - (delta > 0.f ? 1.f : 0.f);
      }
    }
  }
#pragma unroll
  for (int j = 0; j < 8; ++j) {
    float dl[4];
#pragma unroll
    for (int e = 0; e < 4; ++e) {
      const int k = 4 * j + e;
      const float d = N[k] - X[k];                          // signed D^(s+1), Eq. 3
      const float delta = fabsf(fabsf(d) - fabsf(dp[k]));   // |D^(s) - D^(s+1)|
      dp[k] = d;
      dl[e] = delta;
      const float r = (REF_MODE == FITRIG_REF_ABS) ? __saturatef(delta * rcp_approx(fabsf(X[k])))
                                                    : clamped_ratio<REF_MODE>(delta, X[k], C);
      if (j & 1) { S1 += delta; R1 += r; } else { S0 += delta; R0 += r; }
    }
    const float g = fmaxf(fmaxf(dl[0], dl[1]), fmaxf(dl[2], dl[3]));
    if (g > Mx) { Mx = g; jmax = j; }  // strict: keeps the first group in row-major order
  }
  S = S0 + S1;
  R = R0 + R1;
}

// One persistent CTA per SM: warp `ntw` is the producer (one lane issues TMA boxes of ntw adjacent
// tiles into the CTA's ring; full/empty mbarriers), warps 0..ntw-1 are consumers.  A consumer owns
// one 32x32 tile of the box and marches it through time: the two most recent snapshots live in
// registers (A/B ping-pong, no copies), so every snapshot byte is read from HBM once.  The arg-max
// of Delta (R20) is tracked per 16-byte group in the loop; which of its 4 pixels it was is found one
// step later from a 48-byte re-read (3 x cp.async of lines that were fetched moments ago: L2 hits)
// by lane 0, off the critical path.
// UNAL (T = 32, no accumulation): images whose rows do not start on 16-byte boundaries (W % 4 != 0, or an unaligned
// base pointer).  TMA can neither describe such rows (strides must be multiples of 16 bytes) nor start a box off a
// 16-byte boundary, but the stack is ONE contiguous array, and k = 4 / gcd(W, 4) consecutive image rows are a multiple of 16
// bytes: the tensor map describes "super rows" of k image rows (from the base rounded down to 16 bytes, a_off floats
// earlier).  Image row g (counted through the whole stack) is class g % k of super row g / k and starts at element
// (g % k) * W + a_off of it.  The 32 rows of a block are fetched as k boxes of 32 / k rows, one per class, each from the
// 16-byte boundary at or before its rows' first pixel and 4 floats wider: the rows of a class land SHIFTED by
// (class * W + a_off) % 4 floats.  A lane's rows (lane / 8 + 4 j) all belong to one class, so it reads its pixels with
// one base pointer and, depending on the shift, 16-, 8- or 4-byte loads.  Pixels beyond the right / bottom edge are
// not zero-filled by TMA here (the next row / snapshot follows in the super row): the consumer zeroes them.
template <int REF_MODE, bool ACC, int T, bool UNAL = false>
__global__ void __launch_bounds__(32 * (kMaxTilesPerBox + 1), 1)
    tlisi_fused_kernel(const __grid_constant__ CUtensorMap tmap, const FusedParams p) {
  static_assert(!UNAL || !ACC, "the unaligned variant does not accumulate");
  // T >= 8: tiles are lane groups of a warp's block (LaneGeom<T>).  T = 4, 2, 1: a lane holds pixels of several
  // tiles; the block is read with the T = 32 geometry and reduced per 16-byte quad (small_step below).
  constexpr bool kSmall = T < 8;
  constexpr int kLoadGeom = (T == 1) ? 32 : T;  // which pixels a lane holds (lane_row / lane_col)
  using Geo = LaneGeom<(kSmall ? 32 : T)>;
  constexpr int LPT = Geo::LPT, NGRP = 32 / LPT;  // lanes per tile, tiles (lane groups) per warp
  const int acc = ACC ? p.acc : 1;  // ACC = false compiles the accumulation loops away
  extern __shared__ __align__(1024) unsigned char smem[];
  // the shuffle tells the compiler the warp index is warp uniform, so cursors and addresses derived
  // from it live in uniform registers and the vector registers are left to the three tile arrays
  const int warp = __shfl_sync(0xffffffffu, (int)(threadIdx.x >> 5), 0), lane = threadIdx.x & 31;
  const int pitch = p.ntw * 128 + (UNAL ? 16 : 0);  // bytes between rows of a box (UNAL: 4 floats wider, see above)
  const int box_bytes = kFastTile * pitch;
  unsigned char* after_ring = smem + (size_t)p.nstage * box_bytes;
  uint64_t* full = reinterpret_cast<uint64_t*>(after_ring);
  uint64_t* empty = full + kMaxStages;
  // arg-max scratch of this lane's tile (one per lane group)
  float4* scratch = reinterpret_cast<float4*>(after_ring + 2 * kMaxStages * 8) +
                    (warp * NGRP + Geo::sub_row(threadIdx.x & 31) * Geo::NSUB + Geo::sub_col(threadIdx.x & 31)) * kScratchVec;

  if (threadIdx.x == 0) {
    for (int i = 0; i < p.nstage; ++i) {
      mbar_init(smem_u32(&full[i]), 1);
      mbar_init(smem_u32(&empty[i]), p.ntw);
    }
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
  }
  __syncthreads();
  // The first kernel of a call waits for everything ahead of it (the previous call's finalise still reads the records
  // and resets the maximum keys) BEFORE it lets its successors in: a stack b >= 1 of a batch (dep == 2) does not wait at
  // its start, so it may only become schedulable once this grid has seen the previous call complete.
  if (p.dep == 1) pdl_wait();
  pdl_launch_dependents();  // the next kernel of the chain may take its place on the SMs as they fall free

  // this CTA's range of (group, unit) pairs
  const int g_begin = (int)((long long)blockIdx.x * p.G / gridDim.x);
  const int g_end = (int)((long long)(blockIdx.x + 1) * p.G / gridDim.x);
  const uint32_t full_addr = smem_u32(full), empty_addr = smem_u32(empty);

  if (warp == p.ntw) {
    // ---- producer ----
    if (lane == 0) {
      const uint64_t policy = l2_evict_first_policy();
      const uint32_t ring_addr = smem_u32(smem);
      int slot = 0;
      uint32_t phase = 0;
      for (int g = g_begin; g < g_end;) {
        const Segment c = decode_segment(p, g, g_end);
        g += c.nsteps - 2;
        for (int s = 0; s < c.nsteps * acc; ++s) {  // raw snapshots (u0 + step) * acc + i, in order
          mbar_wait(empty_addr + slot * 8, phase ^ 1);  // passes at once on the first lap
          const uint32_t bar = full_addr + slot * 8;
          mbar_arrive_expect_tx(bar, box_bytes);
          if constexpr (UNAL) {
            const int k = p.k_rows, rpc = kFastTile / k;  // rows per class
            const int g0 = ring_slot(p.z0, p.zmask, c.u0 + s) * p.srows + c.ty_local * kFastTile;  // first row of the block
            for (int cls = 0; cls < k; ++cls) {
              const int gf = g0 + ((cls - g0) & (k - 1));  // first row of the block in this class
              const int x = cls * p.W + p.a_off + c.gx * p.ntw * kFastTile;
              tma_load_box2d(ring_addr + slot * box_bytes + cls * rpc * pitch, &tmap, bar, x & ~3, gf / k);
            }
          } else if (p.evict_first)
            tma_load_box_hint(ring_addr + slot * box_bytes, &tmap, bar, c.gx * p.ntw * kFastTile, c.ty_local * kFastTile,
                              ring_slot(p.z0, p.zmask, c.u0 * acc + s), policy);
          else
            tma_load_box(ring_addr + slot * box_bytes, &tmap, bar, c.gx * p.ntw * kFastTile, c.ty_local * kFastTile,
                         ring_slot(p.z0, p.zmask, c.u0 * acc + s));
          if (++slot == p.nstage) { slot = 0; phase ^= 1; }
        }
      }
    }
    return;
  }

  // ---- consumers ----
  const unsigned char* my_col = smem + warp * 128;
  const uint32_t scratch_addr = smem_u32(scratch);
  float A[32], B[32], dp[32];
  float gmax = -3.402823466e38f, zA = 1.f, zB = 1.f;
  int slot = 0;
  uint32_t phase = 0;
  const bool leader = lane == Geo::leader_lane(lane);  // does the bookkeeping of its tile

  // next snapshot of the current segment: box slot -> registers, then hand the slot back
  int zs = 0, seg_ty = 0;      // UNAL: snapshot of the segment the next acquire() takes, and the segment's block row
  int wv = kFastTile, hv = kFastTile;  // UNAL: valid columns / rows of this warp's block
  auto acquire = [&](float (&N)[32], float& zmin) {
    mbar_wait(full_addr + slot * 8, phase);
    if constexpr (UNAL) {
      const int k = p.k_rows, lk = k >> 1;  // k = 1, 2, 4: log2 k = k / 2
      const int g0 = ring_slot(p.z0, p.zmask, zs) * p.srows + seg_ty * kFastTile;
      ++zs;
      const int o0 = g0 & (k - 1);          // the block's first row inside its super row
      const unsigned char* slot_col = smem + (size_t)slot * box_bytes + warp * 128 + lane_col<kLoadGeom>(lane) * 4;
      // where row r of the block sits: class cls = (g0 + r) % k, the ((g0 + r) / k - g0 / k - (cls < o0))-th row of that
      // class's box, shifted by (cls * W + a_off) % 4 floats
      auto row_ptr = [&](int r) {
        const int g = g0 + r, cls = g & (k - 1);
        const int idx = (g >> lk) - (g0 >> lk) - (cls < o0 ? 1 : 0);
        return slot_col + (cls * (kFastTile / k) + idx) * pitch + ((cls * p.W + p.a_off) & 3) * 4;
      };
      // one instruction sequence for all lanes (their shifts differ: a branch per shift would run every variant in
      // turn): 8-byte loads when every shift of this launch is even, 4-byte loads otherwise
      if constexpr (kLoadGeom == 32) {
        // rows lane / 8 + 4 j all belong to one class (4 j is a multiple of k): one pointer, a fixed stride
        const unsigned char* src = row_ptr(lane >> 3);
        const int rstride = (4 / k) * pitch;
        if (p.even_shifts) {
#pragma unroll
          for (int j = 0; j < 8; ++j) {
            const float2 t0 = *reinterpret_cast<const float2*>(src + j * rstride);
            const float2 t1 = *reinterpret_cast<const float2*>(src + j * rstride + 8);
            N[4 * j] = t0.x; N[4 * j + 1] = t0.y; N[4 * j + 2] = t1.x; N[4 * j + 3] = t1.y;
          }
        } else {
#pragma unroll
          for (int j = 0; j < 8; ++j) {
            const float* t = reinterpret_cast<const float*>(src + j * rstride);
            N[4 * j] = t[0]; N[4 * j + 1] = t[1]; N[4 * j + 2] = t[2]; N[4 * j + 3] = t[3];
          }
        }
      } else {
        if (p.even_shifts) {
#pragma unroll
          for (int j = 0; j < 8; ++j) {
            const unsigned char* src = row_ptr(lane_row<kLoadGeom>(lane, j));
            const float2 t0 = *reinterpret_cast<const float2*>(src);
            const float2 t1 = *reinterpret_cast<const float2*>(src + 8);
            N[4 * j] = t0.x; N[4 * j + 1] = t0.y; N[4 * j + 2] = t1.x; N[4 * j + 3] = t1.y;
          }
        } else {
#pragma unroll
          for (int j = 0; j < 8; ++j) {
            const float* t = reinterpret_cast<const float*>(row_ptr(lane_row<kLoadGeom>(lane, j)));
            N[4 * j] = t[0]; N[4 * j + 1] = t[1]; N[4 * j + 2] = t[2]; N[4 * j + 3] = t[3];
          }
        }
      }
      if (wv < kFastTile || hv < kFastTile) {  // (warp uniform) the block hangs over the image edge
        const int c0 = lane_col<kLoadGeom>(lane);
#pragma unroll
        for (int j = 0; j < 8; ++j)
#pragma unroll
          for (int e = 0; e < 4; ++e)
            if (lane_row<kLoadGeom>(lane, j) >= hv || c0 + e >= wv) N[4 * j + e] = 0.f;
      }
    } else {
    load_tile<kLoadGeom>(N, my_col + (size_t)slot * box_bytes, pitch, lane);
    }
    __syncwarp();  // every lane has its copy
    if (lane == 0) mbar_arrive(empty_addr + slot * 8);
    if (++slot == p.nstage) { slot = 0; phase ^= 1; }
    for (int i = 1; i < acc; ++i) {  // accumulation: the image is the sum of acc raw snapshots, added in order
      mbar_wait(full_addr + slot * 8, phase);
      add_tile<kLoadGeom>(N, my_col + (size_t)slot * box_bytes, pitch, lane);
      __syncwarp();
      if (lane == 0) mbar_arrive(empty_addr + slot * 8);
      if (++slot == p.nstage) { slot = 0; phase ^= 1; }
    }
    scan_tile(N, gmax, zmin);
  };
  // a warp whose tile lies beyond the image edge only keeps the ring turning
  auto skip = [&]() {
    mbar_wait(full_addr + slot * 8, phase);
    if (lane == 0) mbar_arrive(empty_addr + slot * 8);
    if (++slot == p.nstage) { slot = 0; phase ^= 1; }
  };

  // ---- one record is always "pending": its arg-max group is known, the pixel inside it is not.
  // Everything the tile's leader lane does costs the whole warp an issue slot, so its path is kept short:
  // the three image pointers of the current unit and the record pointer are carried along incrementally
  // (ip0..ip2, rp below) instead of being rebuilt from indices.  The leader parks the record in the tile's
  // scratch (registers are for the tile arrays): scratch[0 .. 3*acc) the re-read raw pixels of the three
  // images, scratch[kScratchRec] = {sum Delta, max Delta, sum r, group position} (the RawTile layout),
  // scratch[kScratchRec + 1] = {address of the map record}.
  bool pend = false;
  auto resolve_pending = [&]() {  // leader lanes only
    const float4 rec = scratch[kScratchRec];
    RawTile* dst = *reinterpret_cast<RawTile* const*>(&scratch[kScratchRec + 1]);
    cp_async_wait_all();
    float4 img[3];
    const int per_img = (acc <= kMaxAccAsync) ? acc : 1;  // parked quads per image
#pragma unroll
    for (int k = 0; k < 3; ++k) {
      img[k] = scratch[k * per_img];
      if (acc <= kMaxAccAsync) {
        for (int i = 1; i < acc; ++i) {  // the same order of fp32 additions as acquire()
          const float4 t = scratch[k * acc + i];
          img[k].x += t.x; img[k].y += t.y; img[k].z += t.z; img[k].w += t.w;
        }
      }
    }
    const float4 a = img[0], b = img[1], c = img[2];
    const float mx = rec.y;
    // the same three fp32 operations as tile_step -> bit-identical Delta
    const float e0 = fabsf(fabsf(c.x - b.x) - fabsf(b.x - a.x));
    const float e1 = fabsf(fabsf(c.y - b.y) - fabsf(b.y - a.y));
    const float e2 = fabsf(fabsf(c.z - b.z) - fabsf(b.z - a.z));
    const int e = (e0 == mx) ? 0 : (e1 == mx) ? 1 : (e2 == mx) ? 2 : 3;
    float4 o = rec;
    o.w = __int_as_float(__float_as_int(rec.w) + e);
    *reinterpret_cast<float4*>(dst) = o;
  };

  // the unit being finished: its three images at this warp's block origin, and this lane's tile record
  const float* ip0 = p.base;
  const float* ip1 = p.base;
  const float* ip2 = p.base;
  RawTile* rp = p.raw;
  bool tile_exists = true;
  const long long raw_step = (long long)p.Ty * p.Tx;            // records per unit
  const long long img_step = (long long)acc * p.snap_stride;    // elements between consecutive images (plain stack)
  // position of this lane's tile inside the warp's block (0 for T = 32)
  const int sub_off = Geo::sub_row(lane) * T * p.W + Geo::sub_col(lane) * T;

  // reduction of one (tile, unit) over the tile's lane group: exact max + first 16-byte group (one redux pair for a
  // whole-warp tile; a full-mask butterfly over the group's lane bits otherwise -- redux on partial masks would be
  // executed once per group), the two sums by one butterfly (one half of the group carries sum Delta, the other sum r)
  auto finish = [&](float S, float R, float Mx, int jmax) {
    unsigned tmax = __float_as_uint(Mx);  // Mx >= +0: uint order == float order
    unsigned tg = (unsigned)((Geo::row_in_tile(lane) + Geo::RPL * jmax) * T + Geo::col_in_tile(lane));  // row-major in the tile
    if (LPT == 32) {
      const unsigned mbits = tmax;
      tmax = __reduce_max_sync(0xffffffffu, mbits);
      tg = __reduce_min_sync(0xffffffffu, mbits == tmax ? tg : 0x7fffffffu);
    } else {
      auto level = [&](int off) {
        const unsigned om = __shfl_xor_sync(0xffffffffu, tmax, off), op = __shfl_xor_sync(0xffffffffu, tg, off);
        if (om > tmax || (om == tmax && op < tg)) { tmax = om; tg = op; }
      };
      level(Geo::SPLIT);
#pragma unroll
      for (int i = 0; i < Geo::NREST; ++i) level(Geo::rest(i));
    }
    const bool hi = lane & Geo::SPLIT;
    float vsum = (hi ? R : S) + __shfl_xor_sync(0xffffffffu, hi ? S : R, Geo::SPLIT);
#pragma unroll
    for (int i = 0; i < Geo::NREST; ++i) vsum += __shfl_xor_sync(0xffffffffu, vsum, Geo::rest(i));
    const float rsum = __shfl_sync(0xffffffffu, vsum, Geo::leader_lane(lane) | Geo::SPLIT);
    if (leader) {
      if (pend) resolve_pending();
      pend = false;
      if (tile_exists) {  // (tiles of a block that hang over the image edge do not exist)
        scratch[kScratchRec] = make_float4(vsum, __uint_as_float(tmax), rsum, __int_as_float((int)tg));
        *reinterpret_cast<RawTile**>(&scratch[kScratchRec + 1]) = rp;
        // the winning group's 4 pixels in the three images: in bounds (a zero-filled pixel has Delta 0)
        const int off = sub_off + (int)(tg / T) * p.W + (int)(tg % T);
        if constexpr (UNAL) {  // the group is not on a 16-byte boundary and may hang over the right edge (zeroes, as loaded)
          const int col0 = Geo::sub_col(lane) * T + (int)(tg % T);  // column inside the warp's 32 x 32 block
          const float* ip[3] = {ip0, ip1, ip2};
#pragma unroll
          for (int k3 = 0; k3 < 3; ++k3)
#pragma unroll
            for (int e = 0; e < 4; ++e) {
              const bool in = col0 + e < wv;
              cp_async4_zfill(scratch_addr + k3 * 16 + e * 4, in ? ip[k3] + off + e : p.base, in ? 4 : 0);
            }
        } else if (acc <= kMaxAccAsync) {
          for (int i = 0; i < acc; ++i) {
            cp_async16(scratch_addr + i * 16, ip0 + off + i * p.snap_stride);
            cp_async16(scratch_addr + (acc + i) * 16, ip1 + off + i * p.snap_stride);
            cp_async16(scratch_addr + (2 * acc + i) * 16, ip2 + off + i * p.snap_stride);
          }
        } else {  // long accumulations: plain (blocking) loads, L2 hits; the three sums are parked as if acc were 1
          const float* ip[3] = {ip0, ip1, ip2};
#pragma unroll
          for (int k = 0; k < 3; ++k) {
            float4 v = *reinterpret_cast<const float4*>(ip[k] + off);
            for (int i = 1; i < acc; ++i) {
              const float4 t = *reinterpret_cast<const float4*>(ip[k] + off + i * p.snap_stride);
              v.x += t.x; v.y += t.y; v.z += t.z; v.w += t.w;
            }
            scratch[k] = v;
          }
        }
        cp_async_commit();
        pend = true;
      }
    }
    // next unit of the segment (a plain stack: images are img_step apart; the ring mode has one unit per segment)
    ip0 = ip1; ip1 = ip2; ip2 += img_step;
    rp += raw_step;
  };

  // ---- tiles of 4, 2 or 1 pixels: N = x^(s+2), X = x^(s+1) (reference image), dp = signed x^(s+1) - x^(s).  A lane holds
  // whole tiles (lane_row above; T = 1: every pixel is a tile), so there is no reduction across lanes, the first max-Delta
  // pixel (R20) is exact without a re-read, and a lane writes its tiles' records itself (the 8 lanes of a quarter warp
  // write consecutive records: 128 to 512 contiguous bytes).
  int ty0 = 0, tx0 = 0;  // first tile of the warp's block, in tiles
  auto small_step = [&](const float (&N)[32], const float (&X)[32], float (&dq)[32]) {
    const int rq = lane >> 3, cg = lane & 7;
    auto pixel = [&](int k, float& delta, float& r) {
      const float d = N[k] - X[k];                          // signed D^(s+1), Eq. 3
      delta = fabsf(fabsf(d) - fabsf(dq[k]));               // |D^(s) - D^(s+1)|
      dq[k] = d;
      r = clamped_ratio<REF_MODE>(delta, X[k], p.C);        // Eq. 4-5, per pixel (R8 exact)
    };
    if (T == 4) {
#pragma unroll
      for (int h = 0; h < 2; ++h) {  // pixels 16 h .. 16 h + 15 are tile (rq + 4 h, cg) in row-major order
        float S = 0.f, R = 0.f, Mx = -1.f;
        int pos = 0;
#pragma unroll
        for (int k = 0; k < 16; ++k) {
          float delta, r;
          pixel(16 * h + k, delta, r);
          S += delta;
          R += r;
          if (delta > Mx) { Mx = delta; pos = k; }  // strict: the first maximum
        }
        const int ty_r = rq + 4 * h, tx_r = cg;
        if (ty0 + ty_r < p.ty_end && tx0 + tx_r < p.Tx) {
          RawTile o; o.sumD = S; o.maxD = Mx; o.sumR = R; o.pos = pos;
          rp[(long long)ty_r * p.Tx + tx_r] = o;
        }
      }
    } else if (T == 2) {
#pragma unroll
      for (int jp = 0; jp < 4; ++jp) {  // row pair jp: float4 2 jp (upper row) and 2 jp + 1 (lower row)
#pragma unroll
        for (int h = 0; h < 2; ++h) {   // the left / right tile of the quad
          const int k0 = 8 * jp + 2 * h, k1 = k0 + 4;
          float d0, d1, d2, d3, r0, r1, r2, r3;
          pixel(k0, d0, r0); pixel(k0 + 1, d1, r1); pixel(k1, d2, r2); pixel(k1 + 1, d3, r3);
          const float S = ((d0 + d1) + d2) + d3;
          const float R = ((r0 + r1) + r2) + r3;
          float Mx = d0;
          int pos = 0;
          if (d1 > Mx) { Mx = d1; pos = 1; }
          if (d2 > Mx) { Mx = d2; pos = 2; }
          if (d3 > Mx) { Mx = d3; pos = 3; }
          const int ty_r = rq + 4 * jp, tx_r = 2 * cg + h;
          if (ty0 + ty_r < p.ty_end && tx0 + tx_r < p.Tx) {
            RawTile o; o.sumD = S; o.maxD = Mx; o.sumR = R; o.pos = pos;
            rp[(long long)ty_r * p.Tx + tx_r] = o;
          }
        }
      }
    } else {  // T == 1: per-pixel detection; float4 j holds row rq + 4 j, columns 4 cg ..
      // cells of one pixel are kept as 8-byte records {Delta, r} (RawPix; rp - p.raw is a record index); the four
      // records of a quad are 32 contiguous, 16-byte aligned bytes (W % 4 == 0 on this path): two 16-byte stores
      RawPix* const pix = reinterpret_cast<RawPix*>(p.raw) + (rp - p.raw) + 4 * cg;  // (rp is the record of tile (ty0, tx0))
      const int ncol = p.Tx - (tx0 + 4 * cg);  // records of this quad inside the map row (>= 4: all of them)
#pragma unroll
      for (int j = 0; j < 8; ++j) {
        const int row = rq + 4 * j;
        float d0, d1, d2, d3, r0, r1, r2, r3;
        pixel(4 * j, d0, r0); pixel(4 * j + 1, d1, r1); pixel(4 * j + 2, d2, r2); pixel(4 * j + 3, d3, r3);
        if (ncol > 0 && ty0 + row < p.ty_end) {
          RawPix* dst = pix + (long long)row * p.Tx;
          if (!UNAL || (ncol >= 4 && (p.Tx & 1) == 0)) {  // (map rows of even length: the quad's records are 16-byte aligned)
            reinterpret_cast<float4*>(dst)[0] = make_float4(d0, r0, d1, r1);
            reinterpret_cast<float4*>(dst)[1] = make_float4(d2, r2, d3, r3);
          } else {
            RawPix v;
            v.delta = d0; v.r = r0; dst[0] = v;
            if (ncol > 1) { v.delta = d1; v.r = r1; dst[1] = v; }
            if (ncol > 2) { v.delta = d2; v.r = r2; dst[2] = v; }
            if (ncol > 3) { v.delta = d3; v.r = r3; dst[3] = v; }
          }
        }
      }
    }
    rp += raw_step;
  };

  for (int g = g_begin; g < g_end;) {
    const Segment c = decode_segment(p, g, g_end);
    g += c.nsteps - 2;
    const int tx = c.gx * p.ntw + warp;  // this warp's 32x32 block
    if (tx >= p.Tx32) {
      for (int s = 0; s < c.nsteps * acc; ++s) skip();
      continue;
    }
    {
      const long long blk = (long long)(c.ty_local * kFastTile) * p.W + tx * kFastTile;
      ip0 = p.base + blk + (long long)ring_slot(p.z0, p.zmask, c.u0 * acc) * p.snap_stride;
      ip1 = p.base + blk + (long long)ring_slot(p.z0, p.zmask, (c.u0 + 1) * acc) * p.snap_stride;
      ip2 = p.base + blk + (long long)ring_slot(p.z0, p.zmask, (c.u0 + 2) * acc) * p.snap_stride;
      const int ty_t = p.ty_base + c.ty_local * Geo::NSUB + Geo::sub_row(lane);  // tile coordinates in the whole map
      const int tx_t = tx * Geo::NSUB + Geo::sub_col(lane);
      tile_exists = Geo::NSUB == 1 || (ty_t < p.ty_end && tx_t < p.Tx);
      rp = p.raw + ((long long)c.u0 * p.Ty + ty_t) * p.Tx + tx_t;
    }
    if constexpr (UNAL) {
      zs = c.u0; seg_ty = c.ty_local;
      wv = min(kFastTile, p.W - tx * kFastTile);
      hv = min(kFastTile, p.rows - c.ty_local * kFastTile);
    }
    acquire(A, zA);  // x_{u0}
    acquire(B, zB);  // x_{u0+1}
#pragma unroll
    for (int k = 0; k < 32; ++k) dp[k] = B[k] - A[k];
    int step = 2;
    if constexpr (kSmall) {
      constexpr int NS = kFastTile / T;  // tiles per block edge
      ty0 = p.ty_base + c.ty_local * NS;
      tx0 = tx * NS;
      rp = p.raw + ((long long)c.u0 * p.Ty + ty0) * p.Tx + tx0;  // record of the block's first tile
      while (true) {
        acquire(A, zA);
        small_step(A, B, dp);
        if (++step >= c.nsteps) break;
        acquire(B, zB);
        small_step(B, A, dp);
        if (++step >= c.nsteps) break;
      }
    } else {
      while (true) {
        float S, R, Mx;
        int jmax;
        acquire(A, zA);
        tile_step<REF_MODE>(A, B, dp, p.C, __any_sync(0xffffffffu, zB == 0.f), S, R, Mx, jmax);
        finish(S, R, Mx, jmax);
        if (++step >= c.nsteps) break;
        acquire(B, zB);
        tile_step<REF_MODE>(B, A, dp, p.C, __any_sync(0xffffffffu, zA == 0.f), S, R, Mx, jmax);
        finish(S, R, Mx, jmax);
        if (++step >= c.nsteps) break;
      }
    }
  }
  if (leader && pend) resolve_pending();
  // ---- global maximum (a5): zero-filled out-of-bounds pixels are harmless because M >= C > 0 ----
  const unsigned key = __reduce_max_sync(0xffffffffu, float_to_key(gmax));
  if (lane == 0 && g_begin < g_end) atomicMax(p.gmax_key, key);
  if (p.dep == 2) pdl_wait();
}
// ---------------------------------------------------------------------------------------------
// Windows made of cells.  The tLISI kernels reduce square CELLS (the tile itself in the plain case); a window
// is m x m cells, placed every `step` cells:
//   tiles of N_T = 32 * m pixels        cells of 32, step = m   (non-overlapping)
//   overlapping windows (R27, f-4)      cells of `stride` pixels (or 32), step = stride / cell < m
// Sum Delta and sum r add up, max Delta is the max, and the first max-Delta pixel in row-major order OF THE
// WINDOW (R20) is the candidate with the smallest row * N_T + col among the cells that attain the max.
// ---------------------------------------------------------------------------------------------
struct MergeParams {
  const RawTile* cells;  // [U][Cy][Cx]
  RawTile* raw;          // [U][Ty][Tx]
  int U, Ty, Tx, Cy, Cx, m, step, cell, tile;
  int pix8;              // the cells are 8-byte records (cells of one pixel)
};

__global__ void __launch_bounds__(256) merge_cells_kernel(const MergeParams p) {
  pdl_wait();
  const long long n = (long long)p.U * p.Ty * p.Tx;
  // a window of many cells (m * m >= 32) is merged by a whole warp, lanes striding over its cells; a window of a few
  // cells by one thread.  Either way the order of the additions is fixed by the geometry alone: deterministic.
  const bool by_warp = p.m * p.m >= 32;
  const int lane = threadIdx.x & 31;
  const long long tid = (long long)blockIdx.x * blockDim.x + threadIdx.x, nthreads = (long long)gridDim.x * blockDim.x;
  for (long long i = by_warp ? tid / 32 : tid; i < n; i += by_warp ? nthreads / 32 : nthreads) {
    const int u = (int)(i / ((long long)p.Ty * p.Tx));
    const int t = (int)(i - (long long)u * p.Ty * p.Tx);
    const int ty = t / p.Tx, tx = t - ty * p.Tx;
    RawTile o;
    o.sumD = 0.f; o.maxD = -1.f; o.sumR = 0.f; o.pos = 0x7fffffff;
    const int ncell = p.m * p.m;
    for (int k = by_warp ? lane : 0; k < ncell; k += by_warp ? 32 : 1) {
      const int by = k / p.m, bx = k - by * p.m;
      const int cy = ty * p.step + by, cx = tx * p.step + bx;
      if (cy >= p.Cy || cx >= p.Cx) continue;
      const RawTile b = load_raw(p.cells, ((long long)u * p.Cy + cy) * p.Cx + cx, p.pix8);
      o.sumD += b.sumD;
      o.sumR += b.sumR;
      const int pos = (by * p.cell + b.pos / p.cell) * p.tile + bx * p.cell + b.pos % p.cell;
      if (b.maxD > o.maxD || (b.maxD == o.maxD && pos < o.pos)) { o.maxD = b.maxD; o.pos = pos; }
    }
    if (by_warp) {
#pragma unroll
      for (int off = 16; off > 0; off >>= 1) {
        o.sumD += __shfl_xor_sync(0xffffffffu, o.sumD, off);
        o.sumR += __shfl_xor_sync(0xffffffffu, o.sumR, off);
        const float om = __shfl_xor_sync(0xffffffffu, o.maxD, off);
        const int op = __shfl_xor_sync(0xffffffffu, o.pos, off);
        if (om > o.maxD || (om == o.maxD && op < o.pos)) { o.maxD = om; o.pos = op; }
      }
    }
    if (!by_warp || lane == 0) p.raw[i] = o;
  }
}

// ---------------------------------------------------------------------------------------------
// Generic path: any tile size, any width / alignment.  G (power of two <= 32) lanes share one tile.
// ---------------------------------------------------------------------------------------------
struct GenericParams {
  const float* base;        // first snapshot of this launch's rows
  long long snap_stride;    // elements between consecutive snapshots
  int rows;                 // image rows covered by this launch (strip height, or H)
  int W;
  int tile;
  RawTile* raw;
  int Tx, Ty, ty_base, rows_tiles, U;
  int G;                    // lanes per tile
  int z0, zmask;            // real-time mode ring (see FusedParams)
  int acc;                  // snapshot accumulation (see FusedParams)
  int pix8;                 // cells of one pixel: 8-byte records (RawPix)
  float C;
};

template <int REF_MODE>
__global__ void __launch_bounds__(256) tlisi_generic_kernel(const GenericParams p) {
  const int lane = threadIdx.x & 31;
  const int gl = lane & (p.G - 1);
  const long long group = ((long long)blockIdx.x * blockDim.x + threadIdx.x) / p.G;
  const long long per_unit = (long long)p.rows_tiles * p.Tx;
  const long long nitems = per_unit * p.U;
  const bool live = group < nitems;
  float S = 0.f, R = 0.f, Mx = 0.f;
  int pos = 0x7fffffff;
  int u = 0, ty_local = 0, tx = 0;
  if (live) {
    u = (int)(group / per_unit);
    const long long t = group - (long long)u * per_unit;
    ty_local = (int)(t / p.Tx);
    tx = (int)(t - (long long)ty_local * p.Tx);
    const int r0 = ty_local * p.tile, c0 = tx * p.tile;
    const int h = min(p.tile, p.rows - r0), w = min(p.tile, p.W - c0);
    // image k of the unit = sum of raw snapshots (u + k) * acc .. + acc - 1, added in order
    auto image = [&](int k, long long o) {
      float v = p.base[(long long)ring_slot(p.z0, p.zmask, (u + k) * p.acc) * p.snap_stride + o];
      for (int i = 1; i < p.acc; ++i) v += p.base[(long long)ring_slot(p.z0, p.zmask, (u + k) * p.acc + i) * p.snap_stride + o];
      return v;
    };
    bool first = true;
    for (int i = gl; i < h * w; i += p.G) {
      const int r = i / w, c = i - r * w;
      const long long o = (long long)(r0 + r) * p.W + (c0 + c);
      const float a = image(0, o), b = image(1, o), cc = image(2, o);
      const float delta = fabsf(fabsf(b - a) - fabsf(cc - b));
      S += delta;
      if (first || delta > Mx) { Mx = delta; pos = r * p.tile + c; first = false; }
      R += clamped_ratio<REF_MODE>(delta, b, p.C);
    }
  }
  for (int off = p.G >> 1; off > 0; off >>= 1) {
    S += __shfl_xor_sync(0xffffffffu, S, off);
    R += __shfl_xor_sync(0xffffffffu, R, off);
    const float om = __shfl_xor_sync(0xffffffffu, Mx, off);
    const int op = __shfl_xor_sync(0xffffffffu, pos, off);
    if (om > Mx || (om == Mx && op < pos)) { Mx = om; pos = op; }
  }
  if (live && gl == 0) {
    store_raw(p.raw, ((long long)u * p.Ty + (p.ty_base + ty_local)) * p.Tx + tx, p.pix8, S, Mx, R, pos);
  }
}

// ---------------------------------------------------------------------------------------------
// Time-marching kernel for ANY cell size and ANY width / alignment (the generic path).  Same structure as the fused
// kernel -- persistent CTAs, a producer warp that fills a ring of boxes guarded by full / empty mbarriers, every
// snapshot byte read from HBM once, the global maximum folded in -- but nothing is held in registers across time
// steps: the ring keeps the three snapshots of the current unit in shared memory and the consumers read each pixel
// three times from there (shared-memory bandwidth is plentiful), so threads can be mapped to pixels per tile
// geometry at run time:
//   c <= 32  a warp takes floor(32 / c) adjacent tiles at once: lane = column, a loop over the c rows, then a segmented
//            shuffle reduction over each tile's c lanes (consecutive lanes read consecutive words: conflict free)
//   c  > 32  a warp takes one tile, lanes stride over its pixels in row-major order, then a whole-warp butterfly
// A box is nty x ntx whole cells.  Aligned images (16-byte base and strides, W % 4 == 0) are fetched by TMA (box
// coordinates are element-granular, so cell columns need no alignment); anything else by 4-byte cp.async copies
// of the producer warp (zero fill outside the image, completion on the same mbarrier).
// ---------------------------------------------------------------------------------------------
struct MarchParams {
  RawTile* raw;          // [U][Ty][Tx]
  unsigned* gmax_key;
  const float* base;
  long long snap_stride;
  int W, rows;           // image width; rows covered by this launch
  int Tx, Ty, ty_base, ty_end;
  int U;
  int c;                 // cell edge in pixels
  int ntx, nty;          // cells per box
  int bwp, bh;           // box width (floats, a multiple of 4) and height
  int pitch;             // floats between box rows in shared memory: bwp (TMA), or >= bwp + 8 with pitch = W (mod 4) (cp.async)
  int ngx;               // boxes per row of boxes
  int nstage, G;
  int z0, zmask;
  int tma;               // 1: TMA boxes, 0: cp.async copies
  int ncons, nprod;      // consumer and producer warps of this launch
  int dep;               // programmatic dependent launch: as FusedParams::dep
  int pix8;              // cells of one pixel: 8-byte records (RawPix)
  float C;
};

__device__ __forceinline__ void cp_async16_zfill(uint32_t dst, const void* src, int src_bytes) {
  asm volatile("cp.async.cg.shared.global [%0], [%1], 16, %2;" ::"r"(dst), "l"(src), "r"(src_bytes) : "memory");
}
// mbar_wait for the many consumer warps of the generic kernel: a warp that finds the barrier closed sleeps between polls
// (a polling warp takes issue slots from the warps that work; 12 % of all instructions of the cp.async variant were polls)
__device__ __forceinline__ void mbar_wait_sleep(uint32_t bar, uint32_t parity) {
  while (true) {
    uint32_t done;
    asm volatile(
        "{\n\t.reg .pred p;\n\t"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n\t"
        "selp.u32 %0, 1, 0, p;\n\t}"
        : "=r"(done)
        : "r"(bar), "r"(parity)
        : "memory");
    if (done) return;
    __nanosleep(64);
  }
}

// One pixel of a unit: xa, xb, xc = x_s, x_{s+1} (the reference image), x_{s+2}; k = its row-major index in the cell.
// FAST (REF_ABS only): r = sat(Delta * rcp(|x|)) without Eq. 5's "x == 0 -> C" case -- a zero reference pixel then
// yields 1 (Delta > 0) or 0 (sat(NaN), Delta == 0) instead of min(Delta / C, 1); zmin records the smallest |x| seen so
// that the caller can add the difference afterwards (march_zero_fix), which is almost never needed.
template <int REF_MODE, bool FAST>
__device__ __forceinline__ void march_pixel(float xa, float xb, float xc, int k, float C, float& S, float& R, float& Mx, int& mpos,
                                            float& zmin) {
  const float delta = fabsf(fabsf(xb - xa) - fabsf(xc - xb));  // Eq. 3
  S += delta;
  if (FAST) {
    R += __saturatef(delta * rcp_approx(fabsf(xb)));
    zmin = fminf(zmin, fabsf(xb));
  } else {
    R += clamped_ratio<REF_MODE>(delta, xb, C);                  // Eq. 4-5
  }
  if (delta > Mx) { Mx = delta; mpos = k; }                      // strict: the first maximum in ascending k
}
__device__ __forceinline__ float march_zero_fix(float xa, float xb, float xc, float invC) {
  if (xb != 0.f) return 0.f;
  const float delta = fabsf(fabsf(xb - xa) - fabsf(xc - xb));
  return __saturatef(delta * invC) - (delta > 0.f ? 1.f : 0.f);
}

// One whole cell of CS x CS pixels (CS = 0: c_rt x c_rt, loops not unrolled) walked by one lane in row-major order.
template <int REF_MODE, bool FAST, bool FIRST, int CS>
__device__ __forceinline__ void march_tiny_cell(const float* a, const float* b, const float* cv, int pitch, int c_rt, float C,
                                                float& S, float& R, float& Mx, int& mpos, float& zmin, float& gmax) {
  const int c = CS ? CS : c_rt;
  auto row = [&](int rr) {
#pragma unroll
    for (int cc = 0; cc < c; ++cc) {
      const float xa = a[rr * pitch + cc], xb = b[rr * pitch + cc], xc = cv[rr * pitch + cc];
      march_pixel<REF_MODE, FAST>(xa, xb, xc, rr * c + cc, C, S, R, Mx, mpos, zmin);
      gmax = FIRST ? fmaxf(fmaxf(gmax, xc), fmaxf(xa, xb)) : fmaxf(gmax, xc);
    }
  };
  if (CS > 0 && CS <= 7) {  // whole cell unrolled
#pragma unroll
    for (int rr = 0; rr < c; ++rr) row(rr);
  } else {                  // rows unrolled (CS > 0), a loop over the rows
#pragma unroll 1
    for (int rr = 0; rr < c; ++rr) row(rr);
  }
}

struct TagTrue { static constexpr bool value = true; };
struct TagFalse { static constexpr bool value = false; };

template <int REF_MODE, bool SHIFT>
__global__ void __launch_bounds__(32 * kMarchMaxWarps, 1)
    tlisi_march_kernel(const __grid_constant__ CUtensorMap tmap, const MarchParams p) {
  constexpr bool FAST = REF_MODE == FITRIG_REF_ABS;
  extern __shared__ __align__(1024) unsigned char smem[];
  const int warp = __shfl_sync(0xffffffffu, (int)(threadIdx.x >> 5), 0), lane = threadIdx.x & 31;
  const int pitch = p.pitch;  // floats between rows of a box in shared memory
  const int box_floats = p.bh * pitch, box_bytes = box_floats * 4;
  const int slot_bytes = (box_bytes + 127) & ~127;  // TMA destinations are 128-byte aligned
  uint64_t* full = reinterpret_cast<uint64_t*>(smem + (size_t)p.nstage * slot_bytes);
  uint64_t* empty = full + kMaxStages;
  if (threadIdx.x == 0) {
    for (int i = 0; i < p.nstage; ++i) {
      mbar_init(smem_u32(&full[i]), p.tma ? 1 : 32 * p.nprod);
      mbar_init(smem_u32(&empty[i]), p.ncons);
    }
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
  }
  __syncthreads();
  if (p.dep == 1) pdl_wait();  // (before the trigger: see tlisi_fused_kernel)
  pdl_launch_dependents();
  const int g_begin = (int)((long long)blockIdx.x * p.G / gridDim.x);
  const int g_end = (int)((long long)(blockIdx.x + 1) * p.G / gridDim.x);
  const uint32_t full_addr = smem_u32(full), empty_addr = smem_u32(empty), ring_addr = smem_u32(smem);
  // the segment walk of the fused kernel, with boxes of cells: group = box, box-major / time-minor
  auto decode = [&](int g, int& gx, int& gy, int& u0, int& nsteps) {
    const int group = g / p.U;
    u0 = g - group * p.U;
    gy = group / p.ngx;
    gx = group - gy * p.ngx;
    nsteps = min(p.U - u0, g_end - g) + 2;
  };
  // cp.async variant: where the first pixel of a box sits in its 16-byte line of global memory (0..3 floats).  Shared
  // memory takes the box SHIFTED by that much, and its row pitch is congruent to W modulo 4, so that the global and the
  // shared address of every pixel agree modulo 16 bytes: rows travel as 16-byte copies whatever W and the base are.
  auto box_shift = [&](int z, long long org0) {
    return (int)(((uintptr_t)(p.base + (long long)z * p.snap_stride + org0) >> 2) & 3);
  };

  if (warp >= p.ncons) {
    // ---- producers: one lane (TMA), or p.nprod warps that share the rows of a box (cp.async) ----
    const int pw = warp - p.ncons;
    unsigned pos = 0;  // snapshots fetched so far: ring position
    for (int g = g_begin; g < g_end;) {
      int gx, gy, u0, nsteps;
      decode(g, gx, gy, u0, nsteps);
      g += nsteps - 2;
      const int x0 = gx * p.ntx * p.c, y0 = gy * p.nty * p.c;
      for (int s = 0; s < nsteps; ++s, ++pos) {
        const int slot = pos % p.nstage;
        const uint32_t phase = (pos / p.nstage) & 1;
        const int z = ring_slot(p.z0, p.zmask, u0 + s);
        if (p.tma) {
          if (pw == 0 && lane == 0) {
            mbar_wait(empty_addr + slot * 8, phase ^ 1);  // passes at once on the first lap
            mbar_arrive_expect_tx(full_addr + slot * 8, box_bytes);
            tma_load_box(ring_addr + slot * slot_bytes, &tmap, full_addr + slot * 8, x0, y0, z);
          }
        } else {
          // one producer warp polls the barrier, the others sleep at a named barrier until it has passed (polling warps
          // take issue slots from the consumers)
          if (pw == 0) mbar_wait(empty_addr + slot * 8, phase ^ 1);
          asm volatile("bar.sync 1, %0;" ::"r"(32 * p.nprod) : "memory");
          const float* src = p.base + (long long)z * p.snap_stride;
          const int a0 = box_shift(z, (long long)y0 * p.W + x0);
          const uint32_t dst = ring_addr + slot * slot_bytes + a0 * 4;
          const float* aligned_in = reinterpret_cast<const float*>(((uintptr_t)p.base + 15) & ~(uintptr_t)15);
          for (int r = pw; r < p.bh; r += p.nprod) {  // rows of the box, dealt out to the producer warps
            const int y = y0 + r;
            const float* row = src + (long long)y * p.W + x0;
            // up to 3 single floats bring the row to a 16-byte boundary (of global AND shared memory), then 16-byte
            // copies; zero fill outside the image by the source size
            const int head = (4 - (int)(((uintptr_t)row >> 2) & 3)) & 3;
            const int valid = (y < p.rows) ? max(0, min(p.bwp, p.W - x0)) : 0;  // floats of this row inside the image
            const uint32_t drow = dst + r * pitch * 4;
            if (y < p.rows && x0 + p.bwp + 4 <= p.W) {  // the row and its last (overhanging) 16-byte copy lie inside the image row
              if (lane < head) cp_async4_zfill(drow + 4 * lane, row + lane, 4);
              for (int col = head + 4 * lane; col < p.bwp; col += 128) cp_async16(drow + 4 * col, row + col);
            } else {
              if (lane < head) cp_async4_zfill(drow + 4 * lane, lane < valid ? row + lane : src, lane < valid ? 4 : 0);
              for (int col = head + 4 * lane; col < p.bwp; col += 128) {
                const int bytes = max(0, min(16, 4 * (valid - col)));
                cp_async16_zfill(drow + 4 * col, bytes > 0 ? row + col : aligned_in, bytes);
              }
            }
          }
          cp_async_mbar_arrive_noinc(full_addr + slot * 8);  // arrives once this lane's copies have landed
        }
      }
    }
    if (!p.tma) cp_async_wait_all();
    return;
  }

  // ---- consumers ----
  const int c = p.c;
  const bool tiny = c <= kMarchTinyCell;                   // a lane takes a whole tile
  const bool small = c <= 32;
  const int gt = tiny ? 32 : (small ? 32 / c : 1);         // tiles per warp item
  const int ngroups = small ? (p.ntx + gt - 1) / gt : p.ntx;
  const int nitems = p.nty * ngroups;
  const int jt = small ? lane / c : 0, cc0 = small ? lane - jt * c : 0;  // (lanes = columns) this lane's tile in the group, column in it
  const float invC = rcp_approx(p.C);
  float gmax = -3.402823466e38f;
  const long long raw_step = (long long)p.Ty * p.Tx;
  // ring positions of the unit's three snapshots, carried along (no modulo in the loops)
  int sa = 0, sb = (1 % p.nstage), sc = (2 % p.nstage);
  uint32_t pha = 0, phb = (1 / p.nstage) & 1, phc = (2 / p.nstage) & 1;  // parity of the lap each position is in
  auto advance = [&](int& slot, uint32_t& ph) { if (++slot == p.nstage) { slot = 0; ph ^= 1; } };
  // Items are dealt to the warps round-robin over ALL units the CTA walks (item `next` of the running sequence unit 0's
  // items, unit 1's items, ...), not per unit: a box of few items (8 cells of 32 pixels) would leave most warps idle,
  // this way they work on the following units (the ring holds their snapshots already).
  long long next = warp, ubase = 0;
  const unsigned magic = (unsigned)((0x100000000ull + ngroups - 1) / ngroups);  // item / ngroups for item < 2^16
  for (int g = g_begin; g < g_end;) {
    int gx, gy, u0, nsteps;
    decode(g, gx, gy, u0, nsteps);
    g += nsteps - 2;
    const int nunits = nsteps - 2;
    const long long org0 = (long long)(gy * p.nty * p.c) * p.W + gx * p.ntx * p.c;
    // the first two snapshots of the segment
    mbar_wait_sleep(full_addr + sa * 8, pha);
    mbar_wait_sleep(full_addr + sb * 8, phb);
    for (int i = 0; i < nunits; ++i) {
      mbar_wait_sleep(full_addr + sc * 8, phc);
      // the three snapshots of the unit (cp.async variant: each box shifted by the low bits of its global address)
      const float* A = reinterpret_cast<const float*>(smem + (size_t)sa * slot_bytes) +
                       (SHIFT ? box_shift(ring_slot(p.z0, p.zmask, u0 + i), org0) : 0);
      const float* B = reinterpret_cast<const float*>(smem + (size_t)sb * slot_bytes) +
                       (SHIFT ? box_shift(ring_slot(p.z0, p.zmask, u0 + i + 1), org0) : 0);
      const float* Cc = reinterpret_cast<const float*>(smem + (size_t)sc * slot_bytes) +
                        (SHIFT ? box_shift(ring_slot(p.z0, p.zmask, u0 + i + 2), org0) : 0);
      const long long rawu = (long long)(u0 + i) * raw_step;  // first record of the unit
      // The global maximum takes x_{s+2} of every unit and x_s, x_{s+1} of the first unit of a segment: every snapshot of
      // the segment once.  The item loop is compiled twice so that the steady state pays one FMNMX per pixel.
      auto unit_items = [&](auto first_tag) {
      constexpr bool FIRST = decltype(first_tag)::value;
      for (; next < ubase + nitems; next += p.ncons) {
        const int item = (int)(next - ubase);
        const int r = (ngroups == 1) ? item : (int)__umulhi((unsigned)item, magic), gi = item - r * ngroups;
        const int ty = p.ty_base + gy * p.nty + r;
        // Mx starts below every Delta (>= 0), so the first pixel always takes it: no "first" flag in the loops
        float S = 0.f, R = 0.f, Mx = -1.f, zmin = 1.f;
        int mpos = 0;
        if (tiny) {
          // cells of a few pixels: a lane walks ONE whole cell (no reduction across lanes, no idle lanes inside a group of
          // 32 cells); neighbouring lanes are c words apart: conflict free for odd c, two-way for c = 6, 10
          const int tcol = gi * 32 + lane;
          const bool lane_ok = tcol < p.ntx;
          const int org = (r * c) * pitch + (lane_ok ? tcol * c : 0);
          const float* a = A + org;
          const float* b = B + org;
          const float* cv = Cc + org;
          switch (c) {  // the sizes that reach this path (1, 2, 4, 8 ride the fused kernel) are unrolled at compile time
            case 3: march_tiny_cell<REF_MODE, FAST, FIRST, 3>(a, b, cv, pitch, c, p.C, S, R, Mx, mpos, zmin, gmax); break;
            case 5: march_tiny_cell<REF_MODE, FAST, FIRST, 5>(a, b, cv, pitch, c, p.C, S, R, Mx, mpos, zmin, gmax); break;
            case 6: march_tiny_cell<REF_MODE, FAST, FIRST, 6>(a, b, cv, pitch, c, p.C, S, R, Mx, mpos, zmin, gmax); break;
            case 7: march_tiny_cell<REF_MODE, FAST, FIRST, 7>(a, b, cv, pitch, c, p.C, S, R, Mx, mpos, zmin, gmax); break;
            case 9: march_tiny_cell<REF_MODE, FAST, FIRST, 9>(a, b, cv, pitch, c, p.C, S, R, Mx, mpos, zmin, gmax); break;
            case 10: march_tiny_cell<REF_MODE, FAST, FIRST, 10>(a, b, cv, pitch, c, p.C, S, R, Mx, mpos, zmin, gmax); break;
            default: march_tiny_cell<REF_MODE, FAST, FIRST, 0>(a, b, cv, pitch, c, p.C, S, R, Mx, mpos, zmin, gmax); break;
          }
          if (FAST && zmin == 0.f) {  // Eq. 5's x == 0 -> C for this cell's zero reference pixels
            for (int rr = 0; rr < c; ++rr, a += pitch, b += pitch, cv += pitch)
              for (int cc = 0; cc < c; ++cc) R += march_zero_fix(a[cc], b[cc], cv[cc], invC);
          }
          const int tx = gx * p.ntx + tcol;
          if (lane_ok && ty < p.ty_end && tx < p.Tx) {
            store_raw(p.raw, rawu + (long long)ty * p.Tx + tx, p.pix8, S, Mx, R, mpos);
          }
        } else if (small) {
          const int tcol = gi * gt + jt;                    // tile column inside the box
          const bool lane_ok = jt < gt && tcol < p.ntx;
          // lanes without a tile read next to the others (distinct banks), their values go nowhere
          const int col = lane_ok ? tcol * c + cc0 : max(0, min(gi * gt * c + lane, p.bwp - 32 + lane));
          const int org = (r * c) * pitch + col;
          const float* a = A + org;
          const float* b = B + org;
          const float* cv = Cc + org;
#pragma unroll 4
          for (int rr = 0; rr < c; ++rr, a += pitch, b += pitch, cv += pitch) {
            const float xa = *a, xb = *b, xc = *cv;
            march_pixel<REF_MODE, FAST>(xa, xb, xc, rr, p.C, S, R, Mx, mpos, zmin);  // (mpos = the row, for now)
            gmax = FIRST ? fmaxf(fmaxf(gmax, xc), fmaxf(xa, xb)) : fmaxf(gmax, xc);
          }
          if (FAST && zmin == 0.f) {
            a = A + org; b = B + org; cv = Cc + org;
            for (int rr = 0; rr < c; ++rr, a += pitch, b += pitch, cv += pitch) R += march_zero_fix(*a, *b, *cv, invC);
          }
          mpos = mpos * c + cc0;
          // segmented reduction over the c lanes of each tile (fixed tree order: deterministic)
          for (int off = 1; off < c; off <<= 1) {
            const float oS = __shfl_down_sync(0xffffffffu, S, off), oR = __shfl_down_sync(0xffffffffu, R, off);
            const float om = __shfl_down_sync(0xffffffffu, Mx, off);
            const int op = __shfl_down_sync(0xffffffffu, mpos, off);
            if (cc0 + off < c) {
              S += oS; R += oR;
              if (om > Mx || (om == Mx && op < mpos)) { Mx = om; mpos = op; }
            }
          }
          const int tx = gx * p.ntx + tcol;
          if (lane_ok && cc0 == 0 && ty < p.ty_end && tx < p.Tx) {
            store_raw(p.raw, rawu + (long long)ty * p.Tx + tx, p.pix8, S, Mx, R, mpos);
          }
        } else {
          const int tcol = gi;
          const int org = (r * c) * pitch + tcol * c;
          const int n = c * c;
          {
            int o = org + lane, cc = lane;  // c > 32: no wrap needed at the start
#pragma unroll 4
            for (int k = lane; k < n; k += 32) {
              const float xa = A[o], xb = B[o], xc = Cc[o];
              march_pixel<REF_MODE, FAST>(xa, xb, xc, k, p.C, S, R, Mx, mpos, zmin);  // k = row * c + col, ascending per lane
              gmax = FIRST ? fmaxf(fmaxf(gmax, xc), fmaxf(xa, xb)) : fmaxf(gmax, xc);
              cc += 32; o += 32;
              if (cc >= c) { cc -= c; o += pitch - c; }
            }
          }
          if (FAST && zmin == 0.f) {
            int o = org + lane, cc = lane;
            for (int k = lane; k < n; k += 32) {
              R += march_zero_fix(A[o], B[o], Cc[o], invC);
              cc += 32; o += 32;
              if (cc >= c) { cc -= c; o += pitch - c; }
            }
          }
#pragma unroll
          for (int off = 16; off > 0; off >>= 1) {
            S += __shfl_xor_sync(0xffffffffu, S, off);
            R += __shfl_xor_sync(0xffffffffu, R, off);
            const float om = __shfl_xor_sync(0xffffffffu, Mx, off);
            const int op = __shfl_xor_sync(0xffffffffu, mpos, off);
            if (om > Mx || (om == Mx && op < mpos)) { Mx = om; mpos = op; }
          }
          const int tx = gx * p.ntx + tcol;
          if (lane == 0 && ty < p.ty_end && tx < p.Tx) {
            store_raw(p.raw, rawu + (long long)ty * p.Tx + tx, p.pix8, S, Mx, R, mpos);
          }
        }
      }
      };
      if (i == 0) unit_items(TagTrue()); else unit_items(TagFalse());
      ubase += nitems;
      __syncwarp();
      if (lane == 0) mbar_arrive(empty_addr + sa * 8);  // snapshot u0 + i is not needed again
      advance(sa, pha); advance(sb, phb); advance(sc, phc);
    }
    __syncwarp();
    if (lane == 0) {  // the last two snapshots of the segment
      mbar_arrive(empty_addr + sa * 8);
      mbar_arrive(empty_addr + sb * 8);
    }
    advance(sa, pha); advance(sa, pha);
    advance(sb, phb); advance(sb, phb);
    advance(sc, phc); advance(sc, phc);
  }
  const unsigned key = __reduce_max_sync(0xffffffffu, float_to_key(gmax));
  if (lane == 0 && g_begin < g_end) atomicMax(p.gmax_key, key);
  if (p.dep == 2) pdl_wait();
}

// Global maximum over the n pixels of one image (generic path; the fused path folds this into its single
// pass): the image is the sum of `acc` raw snapshots `stride` elements apart, added in order.
__global__ void __launch_bounds__(256) stack_max_kernel(const float* __restrict__ x, long long n, int acc, long long stride,
                                                        unsigned* gmax_key) {
  float m = -3.402823466e38f;
  const long long step = (long long)gridDim.x * blockDim.x;
  for (long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += step) {
    float v = x[i];
    for (int k = 1; k < acc; ++k) v += x[i + k * stride];
    m = fmaxf(m, v);
  }
  const unsigned key = __reduce_max_sync(0xffffffffu, float_to_key(m));
  if ((threadIdx.x & 31) == 0) atomicMax(gmax_key, key);
}

// ---------------------------------------------------------------------------------------------
// Statistics (fp64, deterministic order).  Mean and population standard deviation of a map row from SHIFTED sums:
// with K = the row's first value, d = v - K, a block adds sum d and sum d^2 in a fixed tree order; partials are
// added in chunk order.  mu = K + sum d / n, sigma^2 = sum d^2 / n - (sum d / n)^2.  The shift makes a constant
// row give sigma == 0 exactly (R4) and keeps the subtraction well conditioned (|d| is of the order of sigma).
// ---------------------------------------------------------------------------------------------
struct StatPartial {
  double n, s, s2;  // count, sum d, sum d^2
};

// sum of (a, b) over the block, the same value in every thread; sh: 64 doubles
__device__ __forceinline__ void block_sum2(double& a, double& b, double* sh) {
  for (int off = 16; off > 0; off >>= 1) {
    a += __shfl_xor_sync(0xffffffffu, a, off);
    b += __shfl_xor_sync(0xffffffffu, b, off);
  }
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31, nw = (blockDim.x + 31) >> 5;
  __syncthreads();  // (sh may still be read from a previous use)
  if (lane == 0) { sh[warp] = a; sh[32 + warp] = b; }
  __syncthreads();
  double ta = 0.0, tb = 0.0;
  for (int i = 0; i < nw; ++i) { ta += sh[i]; tb += sh[32 + i]; }  // same order in every thread
  a = ta; b = tb;
}

// Adds the nblk partials of one row in a fixed order (lane-strided, then a shuffle tree) -- one warp.
__device__ __forceinline__ void warp_merge_partials(const StatPartial* parts, int nblk, double& n, double& s, double& s2) {
  const int lane = threadIdx.x & 31;
  n = 0.0; s = 0.0; s2 = 0.0;
  for (int b = lane; b < nblk; b += 32) {
    const volatile StatPartial* sp = parts + b;
    n += sp->n; s += sp->s; s2 += sp->s2;
  }
  for (int off = 16; off > 0; off >>= 1) {
    n += __shfl_xor_sync(0xffffffffu, n, off);
    s += __shfl_xor_sync(0xffffffffu, s, off);
    s2 += __shfl_xor_sync(0xffffffffu, s2, off);
  }
}

__device__ __forceinline__ void stats_from_sums(double K, double n, double s, double s2, double* mu, double* sigma) {
  if (n <= 0.0) { *mu = 0.0; *sigma = 0.0; return; }
  const double m = s / n;
  *mu = K + m;
  *sigma = sqrt(fmax(s2 / n - m * m, 0.0));
}

// The last block of a row to deposit its partial merges them (threadfence + counter).  Called by every thread of the
// block; `sh_flag` is a shared int.
__device__ __forceinline__ void row_stats_finish(StatPartial part, double K, int row, int blk, int nblk, StatPartial* parts,
                                                 unsigned* counters, double* mu, double* sigma, int* sh_flag) {
  if (threadIdx.x == 0) {
    parts[(size_t)row * nblk + blk] = part;
    __threadfence();
    *sh_flag = (atomicAdd(&counters[row], 1u) == (unsigned)nblk - 1);
  }
  __syncthreads();
  if (*sh_flag && threadIdx.x < 32) {
    __threadfence();
    double n, a, b;
    warp_merge_partials(parts + (size_t)row * nblk, nblk, n, a, b);
    if (threadIdx.x == 0) {
      stats_from_sums(K, n, a, b, &mu[row], &sigma[row]);
      counters[row] = 0;  // ready for the next call
    }
  }
  __syncthreads();  // sh_flag is reused by the block's next chunk
}

// ---------------------------------------------------------------------------------------------
// finalize: q, tLISI, per-row statistics (a6, a7).  Map rows are (batch entry, unit) pairs, row = b * U + u.
// ---------------------------------------------------------------------------------------------
constexpr int kFinChunk = 1024;       // map entries per block and pass: at least this many ...
constexpr int kFinLoads = 4;          // records a thread has in flight
constexpr int kFinChunkMax = 16384;   // ... and at most this many (chosen per context from the map size, fitrig_create)

struct FinalizeParams {
  const RawTile* raw;
  float* q;            // [B][U][Ty][Tx]
  float* tlisi;        // context copy
  float* tlisi_user;   // caller's device buffer or NULL
  const unsigned* gmax_key;  // [B] ordered keys of the global maxima
  unsigned* gmax_key_next;   // [B] keys of the NEXT call: zeroed here so that no memset sits in the stream (or NULL)
  float* M_out;        // [B] device scalars: the M that was used
  float M_override;
  float C;
  int H, W, tile, stride, Ty, Tx, U, B;  // windows of `tile` pixels every `stride` pixels (stride == tile: tiles)
  int nblk;            // chunks per row = ceil(Ty * Tx / chunk)
  int chunk;           // map entries per chunk (kFinChunk .. kFinChunkMax, fitrig_create)
  StatPartial* parts;  // [B * U][nblk]
  unsigned* counters;  // [B * U]
  double* mu;          // [B * U]
  double* sigma;       // [B * U]
  // row-shard mode (fitrig_shard_import): M, mu, sigma come from the all-gathered export vectors
  const double* shard_all;  // [shard_world][2 + 2U] or NULL
  int shard_world;
  int user_row;        // -1: tlisi_user is the whole map; r >= 0: tlisi_user is [Ty][Tx] and receives map row r only
  int pix8;            // the map records are 8-byte RawPix (tiles of one pixel)
};

// Eq. 2 / Eq. 6 without the 1 / M^2 factor: p = (sum D / n_t) * max D * (sum r / n_t); n_t = the window's own pixel
// count (R5).  inv_full = 1 / tile^2 serves every full window (a multiplication instead of two fp64 divisions per
// entry, which made the per-pixel maps compute bound); a partial edge window divides by its own count.
__device__ __forceinline__ double tile_product(const RawTile r, int t, int Tx, int H, int W, int tile, int stride,
                                               double inv_full) {
  if (H < 0) return ((double)r.sumD * inv_full) * (double)r.maxD * ((double)r.sumR * inv_full);  // (the caller says: no partial window)
  const int ty = (int)((unsigned)t / (unsigned)Tx), tx = t - ty * Tx;
  const int h = min(tile, H - ty * stride), w = min(tile, W - tx * stride);
  const double inv_n = (h == tile && w == tile) ? inv_full : 1.0 / ((double)h * (double)w);
  return ((double)r.sumD * inv_n) * (double)r.maxD * ((double)r.sumR * inv_n);
}

template <bool PIX8> struct FinRec;  // the record type of the map the finalise reads
template <> struct FinRec<false> {
  typedef RawTile type;
  __device__ static __forceinline__ RawTile widen(const RawTile& r) { return r; }
};
template <> struct FinRec<true> {
  typedef RawPix type;
  __device__ static __forceinline__ RawTile widen(const RawPix& v) {
    RawTile o; o.sumD = v.delta; o.maxD = v.delta; o.sumR = v.r; o.pos = 0;
    return o;
  }
};

// Chan's merge of per-shard (n, mean, M2) triples in shard order
__device__ __forceinline__ void chan_merge(double& n, double& mean, double& m2, double nb, double mb, double m2b) {
  if (nb <= 0.0) return;
  const double tot = n + nb, dlt = mb - mean;
  mean += dlt * (nb / tot);
  m2 += m2b + dlt * dlt * (n * nb / tot);
  n = tot;
}

template <bool PIX8>
__global__ void __launch_bounds__(256, 4) finalize_kernel(const FinalizeParams p) {
  constexpr int kLoads = PIX8 ? 2 * kFinLoads : kFinLoads;  // (8-byte records: twice as many for the same bytes in flight)
  __shared__ double sh[64];
  __shared__ int sh_flag;
  pdl_wait();               // the tLISI kernel's records and its global maximum
  pdl_launch_dependents();  // (a compaction launched behind this kernel waits for its completion all the same)
  const int nt = p.Ty * p.Tx;
  const int R = p.B * p.U;
  const double inv_full = 1.0 / ((double)p.tile * (double)p.tile);
  // no partial window at the bottom / right edge: every entry divides by tile^2 (no index arithmetic per entry)
  const bool all_full = (p.Ty - 1) * p.stride + p.tile <= p.H && (p.Tx - 1) * p.stride + p.tile <= p.W;
  const int Hq = all_full ? -1 : p.H;
  const long long nchunks = (long long)R * p.nblk;
  const int vlen = 2 + 2 * p.U;  // length of one shard's export vector
  for (long long chunk = blockIdx.x; chunk < nchunks; chunk += gridDim.x) {
    const int row = (int)(chunk / p.nblk), blk = (int)(chunk - (long long)row * p.nblk);
    const int b = row / p.U, u = row - b * p.U;
    // M = max(max_s x^(s), C), PAPER.md:223 (R2: signed max), or the caller's override
    float M;
    if (p.shard_all) {
      double m = p.shard_all[0];
      for (int r = 1; r < p.shard_world; ++r) m = fmax(m, p.shard_all[(size_t)r * vlen]);
      M = fmaxf((float)m, p.C);  // the entries are fp32 pixel values: the cast is exact
    } else {
      M = fmaxf(key_to_float(p.gmax_key[b]), p.C);
    }
    if (p.M_override > 0.f) M = p.M_override;
    const double inv_m2 = 1.0 / ((double)M * (double)M);
    const size_t base = (size_t)row * nt;
    // the row's shift: its first q value
    const double K = (double)(float)(tile_product(load_raw(p.raw, base, p.pix8), 0, p.Tx, Hq, p.W, p.tile, p.stride, inv_full) * inv_m2);
    const int begin = blk * p.chunk, end = min(nt, begin + p.chunk);
    double s = 0.0, s2 = 0.0;
    // kFinLoads records per thread are fetched before the first is used (the stores below may alias the loads as far as
    // the compiler knows, so it would not hoist them itself): a big map is a stream, and one record in flight per thread
    // leaves it latency bound
    for (int t0 = begin + threadIdx.x; t0 < end; t0 += kLoads * blockDim.x) {
      typename FinRec<PIX8>::type rec[kLoads];
#pragma unroll
      for (int k = 0; k < kLoads; ++k) {
        const int t = t0 + k * blockDim.x;
        if (t < end) rec[k] = reinterpret_cast<const typename FinRec<PIX8>::type*>(p.raw)[base + t];
      }
#pragma unroll
      for (int k = 0; k < kLoads; ++k) {
        const int t = t0 + k * blockDim.x;
        if (t >= end) break;
        // Eq. 2 / Eq. 6: q = (sum D / n_t) * max D * (sum r / n_t) / M^2, combined in fp64 and rounded once
        const double qd = tile_product(FinRec<PIX8>::widen(rec[k]), t, p.Tx, Hq, p.W, p.tile, p.stride, inv_full) * inv_m2;
        const float qf = (float)qd;
        p.q[base + t] = qf;
        const float tl = (float)(1.0 - qd);
        p.tlisi[base + t] = tl;
        if (p.tlisi_user) {
          if (p.user_row < 0) p.tlisi_user[base + t] = tl;
          else if (row == p.user_row) p.tlisi_user[t] = tl;
        }
        const double d = (double)qf - K;
        s += d;
        s2 += d * d;
      }
    }
    if (p.shard_all) {
      // Eq. 8 over ALL tiles of the image: the shards' (n, mean, M2) of the M-free product p, merged in shard order
      if (blk == 0 && threadIdx.x == 0) {
        double n = 0.0, mean = 0.0, m2 = 0.0;
        for (int r = 0; r < p.shard_world; ++r) {
          const double* v = p.shard_all + (size_t)r * vlen;
          chan_merge(n, mean, m2, v[1], v[2 + u], v[2 + p.U + u]);
        }
        p.mu[row] = mean * inv_m2;
        p.sigma[row] = (n > 0.0) ? sqrt(m2 / n) * inv_m2 : 0.0;
        if (u == 0) p.M_out[b] = M;
      }
      continue;
    }
    if (blk == 0 && u == 0 && threadIdx.x == 0) {
      p.M_out[b] = M;
      if (p.gmax_key_next) p.gmax_key_next[b] = 0u;
    }
    block_sum2(s, s2, sh);
    StatPartial part;
    part.n = (double)(end - begin); part.s = s; part.s2 = s2;
    row_stats_finish(part, K, row, blk, p.nblk, p.parts, p.counters, p.mu, p.sigma, &sh_flag);
  }
}

// ---------------------------------------------------------------------------------------------
// row shards: what the other shards need (fitrig_shard_export): per unit (n, mean, M2) of the M-free product p
// ---------------------------------------------------------------------------------------------
struct ShardExportParams {
  const RawTile* raw;
  const unsigned* gmax_key;
  double* out;          // [2 + 2U]: max pixel, tiles per unit, mean_p[U], M2_p[U]
  int H, W, tile, stride, Ty, Tx, U;
  int nblk, chunk;      // chunks per unit, entries per chunk
  StatPartial* parts;   // [U][nblk]
  unsigned* counters;   // [U]
  int pix8;             // the map records are 8-byte RawPix (tiles of one pixel)
};

__global__ void __launch_bounds__(256) shard_export_kernel(const ShardExportParams p) {
  __shared__ double sh[64];
  __shared__ int sh_flag;
  pdl_wait();
  const int nt = p.Ty * p.Tx;
  const double inv_full = 1.0 / ((double)p.tile * (double)p.tile);
  const long long nchunks = (long long)p.U * p.nblk;
  for (long long chunk = blockIdx.x; chunk < nchunks; chunk += gridDim.x) {
    const int u = (int)(chunk / p.nblk), blk = (int)(chunk - (long long)u * p.nblk);
    const size_t base = (size_t)u * nt;
    const double K = tile_product(load_raw(p.raw, base, p.pix8), 0, p.Tx, p.H, p.W, p.tile, p.stride, inv_full);
    const int begin = blk * p.chunk, end = min(nt, begin + p.chunk);
    double s = 0.0, s2 = 0.0;
    for (int t = begin + threadIdx.x; t < end; t += blockDim.x) {
      const double d = tile_product(load_raw(p.raw, base + t, p.pix8), t, p.Tx, p.H, p.W, p.tile, p.stride, inv_full) - K;
      s += d;
      s2 += d * d;
    }
    block_sum2(s, s2, sh);
    if (threadIdx.x == 0) {
      StatPartial part;
      part.n = (double)(end - begin); part.s = s; part.s2 = s2;
      p.parts[(size_t)u * p.nblk + blk] = part;
      __threadfence();
      sh_flag = (atomicAdd(&p.counters[u], 1u) == (unsigned)p.nblk - 1);
    }
    __syncthreads();
    if (sh_flag && threadIdx.x < 32) {
      __threadfence();
      double n, a, b;
      warp_merge_partials(p.parts + (size_t)u * p.nblk, p.nblk, n, a, b);
      if (threadIdx.x == 0) {
        const double m = (n > 0.0) ? a / n : 0.0;
        p.out[2 + u] = K + m;                                   // mean of p over the shard's tiles
        p.out[2 + p.U + u] = fmax(b - a * m, 0.0);              // M2 = sum (p - mean)^2 = sum d^2 - (sum d)^2 / n
        p.counters[u] = 0;
        if (u == 0) {
          p.out[0] = (double)key_to_float(*p.gmax_key);
          p.out[1] = (double)nt;
        }
      }
    }
    __syncthreads();
  }
}

// ---------------------------------------------------------------------------------------------
// spectrum: per-tile temporal DFT (a10), Eq. 10.  All arithmetic in fp64 (the data is 1 / N_T^2 of the pixels): the
// DC-free series a_u = q_u - mean(q) is a cancellation of values that agree in their first digit or two, so the
// error of eta is what the fp32 q map carries in, amplified by that cancellation, and nothing more.
// ---------------------------------------------------------------------------------------------
struct SpectrumParams {
  const float* q;       // [B][U][nt]
  const double2* tw;    // [U] twiddles (cos, -sin)(2 pi j / U)
  float* eta;           // [B][nt]
  int* kstar;           // [B][nt]
  float* mag;           // [B][U/2][nt] magnitude spectrum
  int harmonics;        // H >= 1: h = harmonic sum over 1, 2, 4, .., H harmonics (R26); 1: maximum magnitude
  int nt;
  int U, B;
  int nblk, chunk;      // chunks per batch entry = ceil(nt / chunk), entries per chunk
  StatPartial* parts;   // [B][nblk]
  unsigned* counters;   // [B]
  double* mu;           // [B]
  double* sigma;        // [B]
  // row shards: the eta statistics come from the all-gathered (n, mean, M2) triples instead (fitrig_shard_import_eta)
  double* shard_out;    // [3] or NULL: this shard's (n, mean, M2) of eta
};

// Magnitude spectrum m_k = |F_k|, k = 1..K, of every tile's DC-free series (Eq. 10): one thread per (tile, block of
// kDftBins bins), tiles fastest so that the loads of q coalesce and the twiddle index is warp uniform (shared-memory
// broadcast).  Direct DFT: the series is short (U = 30 in config 5, 1498 in the paper's real-data run) and of arbitrary
// length (R17).
constexpr int kDftBins = 8;    // bins per thread: every load of q serves this many complex multiply-adds
constexpr int kDftUnroll = 4;  // samples fetched before they are used (the loop is a stream of L2 loads otherwise)

__global__ void __launch_bounds__(128) dft_mag_kernel(const SpectrumParams p) {
  extern __shared__ double2 tws[];  // U twiddles
  pdl_wait();
  pdl_launch_dependents();
  for (int i = threadIdx.x; i < p.U; i += blockDim.x) tws[i] = p.tw[i];
  __syncthreads();
  const long long g = (long long)blockIdx.x * blockDim.x + threadIdx.x;  // (batch entry, tile)
  if (g >= (long long)p.B * p.nt) return;
  const int b = (int)(g / p.nt), t = (int)(g - (long long)b * p.nt);
  const float* q = p.q + (size_t)b * p.U * p.nt + t;
  const int K = p.U / 2, k0 = blockIdx.y * kDftBins + 1;
  // DC removed: a_u = q_u - c.  Any constant c leaves every bin k = 1 .. U-1 unchanged (sum_u e^{-2 pi i k u / U}
  // = 0); the series' mean is the paper's c, its first sample serves the same purpose here -- the q_u agree in their
  // leading digits, so the subtraction keeps the sums well conditioned -- without a pass of its own over the series.
  const double c0 = (double)q[0];
  double re[kDftBins], im[kDftBins];
  int j[kDftBins], kk[kDftBins];  // (k * u) mod U and its step k (0 for bins beyond K: they stay at twiddle 0)
#pragma unroll
  for (int i = 0; i < kDftBins; ++i) { re[i] = 0.0; im[i] = 0.0; j[i] = 0; kk[i] = (k0 + i <= K) ? k0 + i : 0; }
  auto accumulate = [&](double a) {
#pragma unroll
    for (int i = 0; i < kDftBins; ++i) {
      const double2 w = tws[j[i]];
      re[i] = fma(a, w.x, re[i]);
      im[i] = fma(a, w.y, im[i]);
      j[i] += kk[i];              // k <= K < U: one subtraction wraps
      if (j[i] >= p.U) j[i] -= p.U;
    }
  };
  int u = 0;
  for (; u + kDftUnroll <= p.U; u += kDftUnroll) {
    float v[kDftUnroll];
#pragma unroll
    for (int d = 0; d < kDftUnroll; ++d) v[d] = q[(size_t)(u + d) * p.nt];
#pragma unroll
    for (int d = 0; d < kDftUnroll; ++d) accumulate((double)v[d] - c0);
  }
  for (; u < p.U; ++u) accumulate((double)q[(size_t)u * p.nt] - c0);
#pragma unroll
  for (int i = 0; i < kDftBins; ++i)
    if (k0 + i <= K) p.mag[((size_t)b * K + (k0 + i - 1)) * p.nt + t] = (float)sqrt(re[i] * re[i] + im[i] * im[i]);
}

// eta = h(m) per tile (maximum magnitude, or harmonic summing), k*, and the statistics of eta (Eq. 11).
constexpr int kSpecChunk = 256;  // tiles per chunk of the spectrum kernel = its block size

__global__ void __launch_bounds__(kSpecChunk) spectrum_kernel(const SpectrumParams p) {
  __shared__ double sh[64];
  __shared__ int sh_flag;
  __shared__ float sh_e;
  pdl_wait();
  pdl_launch_dependents();
  const int K = p.U / 2;
  const long long nchunks = (long long)p.B * p.nblk;
  for (long long chunk = blockIdx.x; chunk < nchunks; chunk += gridDim.x) {
    const int b = (int)(chunk / p.nblk), blk = (int)(chunk - (long long)b * p.nblk);
    const float* mag = p.mag + (size_t)b * K * p.nt;
    auto eta_of = [&](int t, int* kb_out) {
      float best = 0.f;
      int kb = (K >= 1) ? 1 : 0;
      if (p.harmonics <= 1) {  // h = maximum spectral magnitude, first bin on ties
#pragma unroll 8
        for (int k = 1; k <= K; ++k) {
          const float m = mag[(size_t)(k - 1) * p.nt + t];
          if (k == 1 || m > best) { best = m; kb = k; }
        }
      } else {
        // harmonic summing (R26): s_h(k) = sum_{i<=h} m_{ik} / sqrt(h), h = 1, 2, 4, .., H, h*k <= K
        bool first = true;
        double bestd = 0.0;
        for (int k = 1; k <= K; ++k) {
          double s = 0.0;
          int have = 0;  // harmonics summed so far
          double inv_sqrt_h = 1.0;  // 1 / sqrt(h) for h = 1, 2, 4, ..: times 1 / sqrt(2) per level
          for (int h = 1; h <= p.harmonics && h * k <= K; h *= 2, inv_sqrt_h *= 0.70710678118654752440) {
            for (int i = have + 1; i <= h; ++i) s += (double)mag[(size_t)(i * k - 1) * p.nt + t];  // m_k, m_2k, ... in order
            have = h;
            const double v = s * inv_sqrt_h;
            if (first || v > bestd) { bestd = v; kb = k; first = false; }
          }
        }
        best = (float)bestd;
      }
      *kb_out = kb;
      return best;
    };
    // A chunk is one tile per thread (the work per tile is a loop over the spectrum).  Its statistics are shifted sums
    // around the chunk's OWN first eta (no tile's eta is computed twice), turned into (n, mean, M2); the last block of a
    // stack merges the chunks' triples in chunk order (Chan: exact for a constant map, R4; deterministic).
    const int begin = blk * p.chunk, end = min(p.nt, begin + p.chunk);
    double s = 0.0, s2 = 0.0;
    float e_first = 0.f;
    {
      const int t = begin + threadIdx.x;  // p.chunk <= blockDim.x
      float e = 0.f;
      if (t < end) {
        int kb;
        e = eta_of(t, &kb);
        p.eta[(size_t)b * p.nt + t] = e;
        p.kstar[(size_t)b * p.nt + t] = kb;
      }
      __syncthreads();  // (sh_e may still be read from the previous chunk)
      if (threadIdx.x == 0) sh_e = e;
      __syncthreads();
      e_first = sh_e;
      if (t < end) {
        const double d = (double)e - (double)e_first;
        s = d;
        s2 = d * d;
      }
    }
    block_sum2(s, s2, sh);
    if (threadIdx.x == 0) {
      const double n = (double)(end - begin), m = s / n;
      StatPartial part;
      part.n = n; part.s = (double)e_first + m; part.s2 = fmax(s2 - s * m, 0.0);  // (n, mean, M2)
      p.parts[(size_t)b * p.nblk + blk] = part;
      __threadfence();
      sh_flag = (atomicAdd(&p.counters[b], 1u) == (unsigned)p.nblk - 1);
    }
    __syncthreads();
    if (sh_flag && threadIdx.x == 0) {
      __threadfence();
      double n = 0.0, mean = 0.0, m2 = 0.0;
      for (int c = 0; c < p.nblk; ++c) {
        const volatile StatPartial* sp = p.parts + (size_t)b * p.nblk + c;
        chan_merge(n, mean, m2, sp->n, sp->s, sp->s2);
      }
      if (p.shard_out) { p.shard_out[0] = n; p.shard_out[1] = mean; p.shard_out[2] = m2; }  // one batch entry
      p.mu[b] = mean;                                   // (a shard: its own statistics, until the import)
      p.sigma[b] = (n > 0.0) ? sqrt(m2 / n) : 0.0;
      p.counters[b] = 0;
    }
    __syncthreads();
  }
}

// Global eta statistics from the all-gathered per-shard (n, mean, M2) triples (Chan's merge in shard order).
__global__ void shard_import_eta_kernel(const double* all, int world, double* mu, double* sigma) {
  if (threadIdx.x != 0 || blockIdx.x != 0) return;
  double n = 0.0, mean = 0.0, m2 = 0.0;
  for (int r = 0; r < world; ++r) chan_merge(n, mean, m2, all[3 * r], all[3 * r + 1], all[3 * r + 2]);
  mu[0] = mean;
  sigma[0] = (n > 0.0) ? sqrt(m2 / n) : 0.0;
}

// ---------------------------------------------------------------------------------------------
// compact: z-score, strict threshold, ordered compaction (a8), in ONE pass over the grid: a block counts the candidates
// of its contiguous range of map entries (warp ballot + popc; every warp owns a contiguous part of the range, so there
// is no block barrier per iteration), publishes the count, adds up the published counts of all lower blocks
// (decoupled look-back; blocks take their place in the order from a ticket, so every lower block is running) and writes
// its candidates at that offset, in (row, tile) order.  Blocks without candidates -- almost all -- skip the second
// walk.  The chain is four dependent memory round trips: ticket, entries, publish, look-back.
// ---------------------------------------------------------------------------------------------
struct CompactParams {
  const float* v;       // q [B*U][nt] (image branch) or eta [B][nt] (frequency branch)
  const RawTile* raw;   // image branch: argmax positions
  const int* kstar;     // frequency branch
  const double* mu;     // [rows]
  const double* sigma;  // [rows]
  float tau;
  int rows;             // B*U or B
  int rows_per_batch;   // U or 1
  long long nt;         // tiles per row
  int Tx, Ty, H, W, tile, stride, branch;
  int row_offset;       // image row of this context's first row (row shards), added to y
  int unit_offset;      // real-time mode: index of the unit the one-row map belongs to, added to `snapshot`
  fitrig_candidate* out;
  long long cap;        // device capacity of `out`
  unsigned long long* host_total;  // the count, in mapped pinned host memory
  fitrig_candidate* host_out;      // first host_cap candidates, in mapped pinned host memory
  long long host_cap;
  unsigned long long* host_offsets;  // [B] mapped pinned host memory: candidates that precede stack b (b >= 1; [0] unused)
  int B;
  unsigned long long* status;        // [gridDim.x] (epoch << 32) | count of the block with that ticket
  unsigned* ticket;                  // never reset: every launch draws gridDim.x tickets, the host keeps the running base
  unsigned ticket_base;
  unsigned epoch;                    // launch number, never 0
  long long seg;        // entries per block (multiple of 32 * warps)
  int pix8;             // tiles of one pixel: no position to look up
};

constexpr int kCompactLoads = 8;  // map entries a lane has in flight

// Walks the map entries [b, e) in order -- one warp, all lanes -- and counts (WRITE: also writes, from position
// `running` on) the entries with z > tau.  z of an entry (Eq. 8 on q, R21; sigma == 0 -> z = 0, R4) is formed in fp64,
// rounded to fp32 and compared strictly (R6).  The walk goes row by row: per row, mu, 1 / sigma and a CONSERVATIVE
// fp32 bound thr are set up once (every entry with z > tau has v > thr: thr lies 4e-7 (|mu| + |tau sigma|) below
// mu + tau sigma, far more than the rounding of the fp64 test), so that an entry costs one load and one fp32
// comparison, and only the (rare) survivors of a 32-entry group take the exact test.
// A candidate record from its map entry (row, tile t of the row) and score.
__device__ __forceinline__ fitrig_candidate make_candidate(const CompactParams& p, int row, unsigned t, float z) {
  const long long row_begin = (long long)row * p.nt;
  const int bidx = row / p.rows_per_batch;
  const int ty = (int)(t / (unsigned)p.Tx), tx = (int)(t - (unsigned)ty * (unsigned)p.Tx);
  fitrig_candidate cd;
  if (p.branch == FITRIG_BRANCH_IMAGE) {
    const int pos = p.pix8 ? 0 : p.raw[row_begin + t].pos;  // tile-relative row * N_T + col of the first max-Delta pixel (R20)
    cd.x = tx * p.stride + pos % p.tile;
    cd.y = p.row_offset + ty * p.stride + pos / p.tile;
    cd.snapshot = (row - bidx * p.rows_per_batch) + p.unit_offset;
  } else {
    const int h = min(p.tile, p.H - ty * p.stride), w = min(p.tile, p.W - tx * p.stride);
    cd.x = tx * p.stride + w / 2;  // tile centre (R18)
    cd.y = p.row_offset + ty * p.stride + h / 2;
    cd.snapshot = p.kstar[row_begin + t];
  }
  cd.score = z;
  return cd;
}

constexpr int kCompactStage = 64;  // candidates a warp keeps from its counting pass (more: it walks its range again)
struct StagedCand {
  int row;
  unsigned t;
  float z;
};

// MODE 0: count; 1: count and keep the first kCompactStage candidates in `stage`; 2: write from position `running` on
template <int MODE>
__device__ __forceinline__ unsigned compact_walk(const CompactParams& p, long long b, long long e, int lane,
                                                 unsigned long long running, StagedCand* stage) {
  constexpr bool WRITE = MODE == 2;
  unsigned cnt = 0;
  while (b < e) {
    const int row = (int)(b / p.nt);
    const long long row_begin = (long long)row * p.nt;
    const int n = (int)(min(e, row_begin + p.nt) - b);  // entries of this row in the range
    const double sd = p.sigma[row], mu = p.mu[row];
    const double inv_sigma = (sd > 0.0) ? 1.0 / sd : 0.0;
    float thr;
    if (sd > 0.0) {
      const double ts = (double)p.tau * sd;
      thr = __double2float_rd(mu + ts - 4e-7 * (fabs(mu) + fabs(ts)));
    } else {
      thr = (0.f > p.tau) ? -3.402823466e38f : 3.402823466e38f;  // z == 0 everywhere: all entries, or none
    }
    const float* v = p.v + b;
    const int t0 = (int)(b - row_begin);  // tile index of v[0] inside the row
    for (int c0 = 0; c0 < n; c0 += 32 * kCompactLoads) {
      float vv[kCompactLoads];
#pragma unroll
      for (int k = 0; k < kCompactLoads; ++k) {
        const int o = c0 + 32 * k + lane;
        vv[k] = (o < n) ? v[o] : 0.f;
      }
#pragma unroll
      for (int k = 0; k < kCompactLoads; ++k) {
        const int o = c0 + 32 * k + lane;
        const bool pre = (o < n) && (vv[k] > thr || sd <= 0.0 && 0.f > p.tau);
        if (__ballot_sync(0xffffffffu, pre) == 0u) continue;
        float z = 0.f;
        bool f = false;
        if (pre) {
          z = (float)(((double)vv[k] - mu) * inv_sigma);
          f = z > p.tau;  // strict, R6
        }
        const unsigned bal = __ballot_sync(0xffffffffu, f);
        if (MODE != 0 && f) {
          const unsigned k_in = cnt + __popc(bal & ((1u << lane) - 1u));  // place among this walk's candidates
          const unsigned t = (unsigned)(t0 + o);                          // tile index inside the row (< 2^31)
          if (WRITE) {
            const unsigned long long dst = running + k_in;
            if ((long long)dst < p.cap) {
              const fitrig_candidate cd = make_candidate(p, row, t, z);
              p.out[dst] = cd;
              if ((long long)dst < p.host_cap) p.host_out[dst] = cd;
            }
          } else if (k_in < (unsigned)kCompactStage) {
            StagedCand sc; sc.row = row; sc.t = t; sc.z = z;
            stage[k_in] = sc;
          }
        }
        cnt += __popc(bal);
      }
    }
    b += n;
  }
  return cnt;
}

__global__ void __launch_bounds__(512) compact_kernel(const CompactParams p) {
  __shared__ unsigned warp_cnt[16];
  __shared__ StagedCand s_stage[16][kCompactStage];
  __shared__ unsigned long long s_base;
  __shared__ unsigned s_id;
  pdl_wait();
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31, nw = blockDim.x >> 5;
  // a block's place in the order is the ticket it draws, so a block with a lower place is always already running
  // (block indices carry no such guarantee when other kernels share the device)
  if (threadIdx.x == 0) {
    s_base = 0;
    s_id = atomicAdd(p.ticket, 1u) - p.ticket_base;
  }
  __syncthreads();
  const unsigned id = s_id;
  const long long N = (long long)p.rows * p.nt;
  const long long begin = min(N, (long long)id * p.seg), end = min(N, begin + p.seg);
  const long long wlen = p.seg / nw;  // a multiple of 32
  const long long wb = min(end, begin + warp * wlen), we = min(end, wb + wlen);

  // ---- pass 1: count ----
  const unsigned cnt = compact_walk<1>(p, wb, we, lane, 0ull, s_stage[warp]);
  if (lane == 0) warp_cnt[warp] = cnt;  // (the same in every lane)
  __syncthreads();
  unsigned before = 0, total = 0;
  for (int w = 0; w < nw; ++w) {
    const unsigned cw = warp_cnt[w];
    if (w < warp) before += cw;
    total += cw;
  }
  // ---- publish, then add up the counts of all lower blocks ----
  if (threadIdx.x == 0)
    *reinterpret_cast<volatile unsigned long long*>(p.status + id) = ((unsigned long long)p.epoch << 32) | total;
  unsigned long long below = 0;
  for (long long j = (long long)id - 1 - threadIdx.x; j >= 0; j -= blockDim.x) {
    unsigned long long v;
    do {
      v = *reinterpret_cast<volatile unsigned long long*>(p.status + j);
    } while ((unsigned)(v >> 32) != p.epoch);
    below += (unsigned)v;
  }
  for (int off = 16; off > 0; off >>= 1) below += __shfl_xor_sync(0xffffffffu, below, off);
  if (lane == 0 && below) atomicAdd(&s_base, below);
  __syncthreads();
  const unsigned long long base = s_base;
  if (threadIdx.x == 0 && id == gridDim.x - 1) *p.host_total = base + total;
  // ---- stacks of a batch: how many candidates precede the first entry of stack b (the host takes differences) ----
  if (p.B > 1 && warp == 0) {
    const long long per = (long long)p.rows_per_batch * p.nt;  // entries per stack
    for (long long b = (begin + per - 1) / per; b < p.B && b * per < end; ++b) {
      if (b == 0) continue;
      const long long edge = b * per;  // begin <= edge < end
      unsigned long long c = base;
      for (int w = 0; w < nw; ++w) {   // whole warps below the edge, then a recount inside the one that holds it
        const long long swb = min(end, begin + w * wlen), swe = min(end, swb + wlen);
        if (swe <= edge) { c += warp_cnt[w]; continue; }
        if (swb >= edge) break;
        c += compact_walk<0>(p, swb, edge, lane, 0ull, nullptr);
        break;
      }
      if (lane == 0) p.host_offsets[b] = c;
    }
  }
  // ---- write in order: the candidates kept from the counting pass, or -- a warp with more of them than it could keep --
  // a second walk
  if (cnt > (unsigned)kCompactStage) {
    compact_walk<2>(p, wb, we, lane, base + before, nullptr);
  } else {
    for (unsigned k = lane; k < cnt; k += 32) {
      const unsigned long long dst = base + before + k;
      if ((long long)dst < p.cap) {
        const StagedCand sc = s_stage[warp][k];
        const fitrig_candidate cd = make_candidate(p, sc.row, sc.t, sc.z);
        p.out[dst] = cd;
        if ((long long)dst < p.host_cap) p.host_out[dst] = cd;
      }
    }
  }
}

// ---------------------------------------------------------------------------------------------
// Sub-tile localisation by interpolating eta (reading R28 in DESIGN.md): the spectrum matrix is a
// sample of a surface at the tile centres (index coordinates: tile column tx at u = tx); the surface is the tensor
// product -- along x in every tile row, then along y -- of one of the four named 1-D schemes; for a selected tile it
// is evaluated on a lattice of 1 / oversample pixels within one tile of the tile's centre (clipped to the hull of the
// centres) and the position is the first maximum in row-major order.  fp64 throughout (a few thousand operations per
// candidate).  spline_rows_kernel: one thread per tile row solves that row's not-a-knot spline.  localise_kernel: one
// CTA per candidate, one thread per lattice column: the column of row-interpolant values at its u (all Ty rows: the
// spline is global), that column's own spline, the best lattice row; then the first maximum over the columns.
// ---------------------------------------------------------------------------------------------
// Second derivatives of the not-a-knot cubic spline through (i, f_i), unit spacing.  With equal spacing the end
// condition m_0 - 2 m_1 + m_2 = 0 turns the first interior equation into m_1 = d_1 (d_i = f_{i-1} - 2 f_i + f_{i+1}),
// likewise m_{n-2} = d_{n-2}; the rest is the (1, 4, 1) system for m_2 .. m_{n-3} (Thomas), then m_0 = 2 m_1 - m_2 and
// m_{n-1} = 2 m_{n-2} - m_{n-3}.  f and m may have any stride; cp: n doubles of scratch.
__device__ inline void spline_nak(const double* f, int fs, int n, double* m, int ms, double* cp, int cs) {
  if (n < 3) {
    for (int i = 0; i < n; ++i) m[i * ms] = 0.0;
    return;
  }
  auto d = [&](int i) { return f[(i - 1) * fs] - 2.0 * f[i * fs] + f[(i + 1) * fs]; };
  if (n == 3) {
    m[0] = m[ms] = m[2 * ms] = d(1);
    return;
  }
  m[ms] = d(1);
  m[(n - 2) * ms] = d(n - 2);
  if (n > 4) {
    // unknowns k = 2 .. n-3; forward sweep stores the modified right-hand side in m, the modified diagonal in cp
    double cprev = 0.0, dprev = 0.0;
    for (int k = 2; k <= n - 3; ++k) {
      double rhs = 6.0 * d(k);
      if (k == 2) rhs -= m[ms];
      if (k == n - 3) rhs -= m[(n - 2) * ms];
      const double den = 4.0 - ((k == 2) ? 0.0 : cprev);
      cprev = 1.0 / den;
      dprev = (rhs - ((k == 2) ? 0.0 : dprev)) / den;
      cp[k * cs] = cprev;
      m[k * ms] = dprev;
    }
    for (int k = n - 4; k >= 2; --k) m[k * ms] -= cp[k * cs] * m[(k + 1) * ms];
  }
  m[0] = 2.0 * m[ms] - m[2 * ms];
  m[(n - 1) * ms] = 2.0 * m[(n - 2) * ms] - m[(n - 3) * ms];
}

struct Interp1 {
  // value at u in [0, n-1] of the 1-D interpolant through (i, f[i * fs]); m: spline second derivatives (stride ms)
  __device__ static double keys_w(double s) {  // Keys (1981), a = -1/2
    s = fabs(s);
    if (s <= 1.0) return (1.5 * s - 2.5) * s * s + 1.0;
    if (s < 2.0) return ((-0.5 * s + 2.5) * s - 4.0) * s + 2.0;
    return 0.0;
  }
  __device__ static double sample(const double* f, int fs, int n, int i) {  // Keys' boundary samples
    if (i >= 0 && i < n) return f[i * fs];
    if (n == 2) return (i < 0) ? 2.0 * f[0] - f[fs] : 2.0 * f[fs] - f[0];
    return (i < 0) ? 3.0 * f[0] - 3.0 * f[fs] + f[2 * fs]
                   : 3.0 * f[(n - 1) * fs] - 3.0 * f[(n - 2) * fs] + f[(n - 3) * fs];
  }
  __device__ static double diff(const double* f, int fs, int n, int i) {  // f_{i+1} - f_i, extended linearly twice
    if (i >= 0 && i <= n - 2) return f[(i + 1) * fs] - f[i * fs];
    if (i < 0) {
      const double d0 = f[fs] - f[0], d1 = f[2 * fs] - f[fs];
      const double a = 2.0 * d0 - d1;
      return (i == -1) ? a : 2.0 * a - d0;
    }
    const double e0 = f[(n - 1) * fs] - f[(n - 2) * fs], e1 = f[(n - 2) * fs] - f[(n - 3) * fs];
    const double a = 2.0 * e0 - e1;
    return (i == n - 1) ? a : 2.0 * a - e0;
  }
  __device__ static double makima_slope(const double* f, int fs, int n, int i) {
    const double a = diff(f, fs, n, i - 2), b = diff(f, fs, n, i - 1), c = diff(f, fs, n, i), e = diff(f, fs, n, i + 1);
    const double w1 = fabs(e - c) + fabs(e + c) / 2.0, w2 = fabs(b - a) + fabs(b + a) / 2.0;
    return (w1 + w2 > 0.0) ? (w1 * b + w2 * c) / (w1 + w2) : 0.0;
  }
  __device__ static double eval(const double* f, int fs, const double* m, int ms, int n, int method, double u) {
    if (n == 1) return f[0];
    int i = (int)floor(u);
    i = max(0, min(i, n - 2));
    const double t = u - (double)i;
    if (method == FITRIG_INTERP_BILINEAR || n == 2) return (1.0 - t) * f[i * fs] + t * f[(i + 1) * fs];
    if (method == FITRIG_INTERP_BICUBIC) {
      double s = 0.0;
      for (int k = -1; k <= 2; ++k) s += sample(f, fs, n, i + k) * keys_w(t - (double)k);
      return s;
    }
    if (method == FITRIG_INTERP_SPLINE) {
      const double a = 1.0 - t;
      return a * f[i * fs] + t * f[(i + 1) * fs] + ((a * a * a - a) * m[i * ms] + (t * t * t - t) * m[(i + 1) * ms]) / 6.0;
    }
    const double s0 = makima_slope(f, fs, n, i), s1 = makima_slope(f, fs, n, i + 1);
    const double t2 = t * t, t3 = t2 * t;
    return (2.0 * t3 - 3.0 * t2 + 1.0) * f[i * fs] + (t3 - 2.0 * t2 + t) * s0 + (-2.0 * t3 + 3.0 * t2) * f[(i + 1) * fs] +
           (t3 - t2) * s1;
  }
};

struct LocaliseParams {
  const double* eta;    // [Ty][Tx]
  double* rowm;         // [Ty][Tx] second derivatives of the row splines (spline only)
  double* scratch;      // [Ty][Tx] (spline_rows_kernel) / per candidate [3][side][Ty] (localise_kernel)
  const int2* tiles;    // [n] (tx, ty) of the selected tiles
  fitrig_position* out; // [n]
  int n, Ty, Tx, tile, method, oversample;
};

__global__ void spline_rows_kernel(const LocaliseParams p) {
  const int r = blockIdx.x * blockDim.x + threadIdx.x;
  if (r >= p.Ty) return;
  spline_nak(p.eta + (size_t)r * p.Tx, 1, p.Tx, p.rowm + (size_t)r * p.Tx, 1, p.scratch + (size_t)r * p.Tx, 1);
}

__global__ void __launch_bounds__(128) localise_kernel(const LocaliseParams p) {
  __shared__ double s_val[128];
  __shared__ int s_j[128], s_i[128];
  const int k = blockIdx.x;
  const int tx = p.tiles[k].x, ty = p.tiles[k].y;
  const int half = p.tile * p.oversample, side = 2 * half + 1;
  // per candidate scratch: col, colm, cp, each [side][Ty] with the lattice column fastest (coalesced across threads)
  double* col = p.scratch + (size_t)k * 3 * side * p.Ty;
  double* colm = col + (size_t)side * p.Ty;
  double* cp = colm + (size_t)side * p.Ty;
  double best = 0.0;
  int bj = 0x7fffffff, bi = 0x7fffffff;
  for (int ii = threadIdx.x; ii < side; ii += blockDim.x) {  // lattice columns, ascending per thread
    const int i = ii - half;
    const double u = (double)tx + (double)i / (double)half;
    if (u < 0.0 || u > (double)(p.Tx - 1)) continue;
    for (int r = 0; r < p.Ty; ++r)
      col[(size_t)r * side + ii] = Interp1::eval(p.eta + (size_t)r * p.Tx, 1, p.rowm + (size_t)r * p.Tx, 1, p.Tx, p.method, u);
    if (p.method == FITRIG_INTERP_SPLINE) spline_nak(col + ii, side, p.Ty, colm + ii, side, cp + ii, side);
    for (int j = -half; j <= half; ++j) {
      const double v = (double)ty + (double)j / (double)half;
      if (v < 0.0 || v > (double)(p.Ty - 1)) continue;
      const double val = Interp1::eval(col + ii, side, colm + ii, side, p.Ty, p.method, v);
      // first maximum in (j, i) order: this thread walks i ascending, j ascending
      if (bj == 0x7fffffff || val > best || (val == best && (j < bj || (j == bj && i < bi)))) { best = val; bj = j; bi = i; }
    }
  }
  s_val[threadIdx.x] = best; s_j[threadIdx.x] = bj; s_i[threadIdx.x] = bi;
  __syncthreads();
  if (threadIdx.x == 0) {
    for (int t = 1; t < (int)blockDim.x; ++t) {
      if (s_j[t] == 0x7fffffff) continue;
      if (bj == 0x7fffffff || s_val[t] > best || (s_val[t] == best && (s_j[t] < bj || (s_j[t] == bj && s_i[t] < bi)))) {
        best = s_val[t]; bj = s_j[t]; bi = s_i[t];
      }
    }
    const double xc = ((double)tx + 0.5) * (double)p.tile - 0.5, yc = ((double)ty + 0.5) * (double)p.tile - 0.5;
    fitrig_position o;
    o.x = xc + (double)bi / (double)p.oversample;
    o.y = yc + (double)bj / (double)p.oversample;
    o.value = best;
    p.out[k] = o;
  }
}

// ---------------------------------------------------------------------------------------------
// Stopping rule of snapshot accumulation (reading R30): for a group size g, the contrast of adjacent
// accumulated snapshots d(g) = mean |A_{j+1} - A_j| / mean |A_j|.  accum_contrast_kernel: a thread walks its pixels
// (grid stride) through the J = L / g accumulated snapshots (A_j summed in fp32 in snapshot order, as the tLISI kernels
// accumulate), keeps sum |A_{j+1} - A_j| and sum |A_j| in fp64; block partials in block order.  accum_choose_kernel:
// one block adds the partials of every level in a fixed order, forms d, and takes the first level with d >= eps (else
// the last level).  Every snapshot byte is read once per level.
// ---------------------------------------------------------------------------------------------
constexpr int kAccumLevels = 6;  // g = 1, 2, 4, 8, 16, 32

struct AccumChoice {
  int g;                        // the chosen group size
  int n_levels;                 // levels looked at
  double contrast[kAccumLevels];
};

__global__ void __launch_bounds__(256) accum_contrast_kernel(const float* __restrict__ x, long long hw, int L, int g, double2* partials) {
  __shared__ double sh[64];
  const int J = L / g;
  double num = 0.0, den = 0.0;
  const long long step = (long long)gridDim.x * blockDim.x;
  for (long long p = (long long)blockIdx.x * blockDim.x + threadIdx.x; p < hw; p += step) {
    float prev = 0.f;
    for (int j = 0; j < J; ++j) {
      const float* s = x + (long long)j * g * hw + p;
      float a = s[0];
      for (int i = 1; i < g; ++i) a += s[(long long)i * hw];  // A_j: g raw snapshots added in order
      if (j > 0) num += (double)fabsf(a - prev);                // Eq. 3 on accumulated snapshots
      den += (double)fabsf(a);
      prev = a;
    }
  }
  block_sum2(num, den, sh);
  if (threadIdx.x == 0) partials[blockIdx.x] = make_double2(num, den);
}

__global__ void __launch_bounds__(256) accum_choose_kernel(const double2* partials, int nblocks, int n_levels, int L, long long hw,
                                                           float eps, AccumChoice* out) {
  __shared__ double sh[64];
  int chosen = -1;
  for (int lv = 0; lv < n_levels; ++lv) {
    double num = 0.0, den = 0.0;
    for (int b = threadIdx.x; b < nblocks; b += blockDim.x) {
      const double2 v = partials[(size_t)lv * nblocks + b];
      num += v.x;
      den += v.y;
    }
    block_sum2(num, den, sh);
    const int J = L / (1 << lv);
    const double mn = num / ((double)(J - 1) * (double)hw), md = den / ((double)J * (double)hw);
    const double d = (md > 0.0) ? mn / md : 0.0;
    if (threadIdx.x == 0) out->contrast[lv] = d;
    if (chosen < 0 && d >= (double)eps) chosen = lv;  // (the same value in every thread)
  }
  if (threadIdx.x == 0) {
    // progressive combination stops at the first level that reaches eps: later levels are reported as not looked at
    out->n_levels = (chosen < 0) ? n_levels : chosen + 1;
    out->g = 1 << ((chosen < 0) ? n_levels - 1 : chosen);
  }
}

// ---------------------------------------------------------------------------------------------
// calibration: what a plain read-only stream of the same buffer achieves on this device (fitrig_probe_read_bandwidth).
// The roofline denominator of MEASURED_PEAKS.json is a COPY (read + write); a read-only kernel can exceed it.
// ---------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(512) read_probe_kernel(const float4* __restrict__ x, long long n4, float* sink) {
  float m = -3.402823466e38f;
  const long long step = (long long)gridDim.x * blockDim.x;
  long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  for (; i + 3 * step < n4; i += 4 * step) {  // four independent 16-byte loads in flight per thread
    const float4 a = x[i], b = x[i + step], c = x[i + 2 * step], d = x[i + 3 * step];
    m = fmaxf(m, fmaxf(fmaxf(fmaxf(a.x, a.y), fmaxf(a.z, a.w)), fmaxf(fmaxf(b.x, b.y), fmaxf(b.z, b.w))));
    m = fmaxf(m, fmaxf(fmaxf(fmaxf(c.x, c.y), fmaxf(c.z, c.w)), fmaxf(fmaxf(d.x, d.y), fmaxf(d.z, d.w))));
  }
  for (; i < n4; i += step) {
    const float4 a = x[i];
    m = fmaxf(m, fmaxf(fmaxf(a.x, a.y), fmaxf(a.z, a.w)));
  }
  if (m == 1.2345e-30f) *sink = m;  // keeps the loads alive; practically never true
}

}  // namespace fitrig
