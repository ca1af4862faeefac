"""CPU tier: the C-ABI library loads without a GPU and exports every symbol include/fitrig.h declares;
host-only entry points (plan query, argument validation) behave as the header says."""
import ctypes

import pytest

import paper_2509_21754_b200 as fitrig
from paper_2509_21754_b200 import binding


def test_library_loads_and_exports_every_declared_symbol():
    L = fitrig.load_library()
    names = fitrig.exported_symbols()
    assert {"fitrig_create", "fitrig_tlisi", "fitrig_detect", "fitrig_stream"} <= set(names)
    for n in names:
        assert hasattr(L, n), f"{n} declared in include/fitrig.h but not exported"
    assert fitrig.version().startswith("fitrig-b200")
    assert isinstance(fitrig.last_error(), str)


def test_struct_layouts_match_header():
    assert ctypes.sizeof(binding._Candidate) == 16  # "16 bytes" in fitrig.h
    assert ctypes.sizeof(binding._Params) == 64
    assert binding.CANDIDATE_DTYPE.itemsize == 16


def test_plan_query_tile_grid_and_partial_tiles():
    p = fitrig.plan_query(50000, 50000, 4)
    assert (p.units, p.Ty, p.Tx) == (2, 1563, 1563)  # ceil(50000/32), R5
    assert p.path == 0 and p.strip_rows % 32 == 0 and p.n_strips * p.strip_rows >= 50000
    p = fitrig.plan_query(250, 250, 8, tile=8)
    # W % 4 != 0: rows off 16-byte boundaries ride the fused kernel through super rows of k = 2 image rows (8 * 250 rows: even)
    assert (p.units, p.Ty, p.Tx, p.path) == (6, 32, 32, 0) and p.box_tiles <= 7
    p = fitrig.plan_query(250, 252, 8, tile=8)
    assert (p.Ty, p.Tx, p.path) == (32, 32, 0) and p.strip_rows % 32 == 0  # N_T = 8, 16 ride the fused kernel
    assert fitrig.plan_query(250, 252, 8, tile=16).path == 0
    assert fitrig.plan_query(250, 252, 8, tile=64).path == 0 and fitrig.plan_query(250, 252, 8, tile=96).path == 0  # 32 * m
    assert fitrig.plan_query(250, 252, 8, tile=5).path == 1 and fitrig.plan_query(250, 252, 8, tile=7).path == 1
    # tiles with a divisor of 16, 8 or 4 pixels are m x m cells of that size on the fused kernel
    assert all(fitrig.plan_query(250, 252, 8, tile=t).path == 0 for t in (12, 24, 48, 100))
    assert all(fitrig.plan_query(250, 252, 8, tile=t).path == 0 for t in (1, 2, 4))  # tiles inside a lane's quads
    p = fitrig.plan_query(256, 250, 8)
    assert p.path == 0 and p.box_tiles <= 7  # W % 4 != 0: super rows; a TMA box holds at most 256 elements, 4 of them are slack
    assert fitrig.plan_query(33, 251, 5).path == 1   # 5 * 33 rows are not a multiple of k = 4: the generic kernel
    assert fitrig.plan_query(33, 251, 8).path == 0
    assert fitrig.plan_query(256, 250, 8, tile=5).path == 1 and fitrig.plan_query(256, 250, 8, accumulate=2).path == 1
    p = fitrig.plan_query(256, 252, 8)
    assert p.path == 0 and p.Tx == 8


def test_plan_query_balances_units_over_ctas():
    # 64 x 8 boxes of 8 tiles x 62 units on 148 SMs: every CTA gets ceil(31744 / 148) = 215 (box, unit) pairs
    p = fitrig.plan_query(2048, 2048, 64, num_sms=148)
    assert p.box_tiles == 8 and p.warps_per_cta == 9 and p.grid == 148 and p.units_per_cta == 215
    assert p.smem_bytes <= 227 * 1024 and p.stages >= 4
    # tiny problem (64 tiles x 6 units): narrow boxes, spread thin so that the GPU is not left to a few SMs
    p = fitrig.plan_query(256, 256, 8, num_sms=148)
    assert p.grid >= 96 and p.units_per_cta >= 2 and p.box_tiles < 8
    # one tile, one unit
    p = fitrig.plan_query(32, 32, 3, num_sms=148)
    assert p.grid == 1 and p.box_tiles == 1 and p.warps_per_cta == 2 and p.units_per_cta == 1
    # 50000 wide: 1563 tiles = 195 boxes of 8 + one of 3 (the rest of the last box is zero-filled by TMA)
    p = fitrig.plan_query(50000, 50000, 4, num_sms=148)
    assert p.box_tiles == 8 and p.grid == 148


@pytest.mark.parametrize("H,W,L,kw", [
    (0, 16, 3, {}), (16, 0, 3, {}), (16, 16, 2, {}),  # R10: L < 3
    (16, 16, 3, {"tile": -1}), (16, 16, 3, {"ref_mode": 7}), (16, 16, 3, {"branch": 2}),
    (64, 64, 3, {"tile": 32, "strip_rows": 48}),  # not a multiple of tile
    (16, 16, 3, {"C": 1e-35}),
])
def test_invalid_arguments_are_rejected_before_any_cuda_call(H, W, L, kw):
    with pytest.raises(fitrig.FitrigError) as e:
        fitrig.plan_query(H, W, L, **kw)
    assert e.value.code == binding.ERR_INVALID_ARG
    with pytest.raises(fitrig.FitrigError) as e:
        fitrig.Context(H, W, L, **kw)
    assert e.value.code == binding.ERR_INVALID_ARG


def test_no_cpu_fallback_without_a_device():
    import torch
    if torch.cuda.is_available():
        pytest.skip("a CUDA device is present")
    with pytest.raises(fitrig.FitrigError) as e:
        fitrig.Context(64, 64, 4)
    assert e.value.code == binding.ERR_CUDA  # fails loudly; nothing routes to the oracle


def test_header_is_plain_c_and_links_from_c(tmp_path):
    """include/fitrig.h must compile as C99 (no C++, no torch types) and the host-only entry points must be
    callable from a C program linked against the in-tree library."""
    import os
    import subprocess
    root = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
    src = tmp_path / "abi.c"
    src.write_text(r'''
#include <stdio.h>
#include <string.h>
#include "fitrig.h"
int main(void) {
  fitrig_params p;
  fitrig_plan plan;
  memset(&p, 0, sizeof p);
  if (sizeof(fitrig_candidate) != 16 || sizeof(fitrig_params) != 64) return 2;
  if (fitrig_plan_query(50000, 50000, 4, &p, 148, &plan) != FITRIG_OK) return 3;
  if (plan.Ty != 1563 || plan.Tx != 1563 || plan.units != 2) return 4;
  p.tile = -1;
  if (fitrig_plan_query(64, 64, 8, &p, 0, &plan) != FITRIG_ERR_INVALID_ARG) return 5;
  printf("%s\n", fitrig_version());
  return 0;
}
''')
    exe = tmp_path / "abi"
    lib_dir = os.path.dirname(fitrig.lib_path())
    subprocess.run(["gcc", "-std=c99", "-Wall", "-Werror", "-pedantic", "-I", os.path.join(root, "include"), str(src),
                    "-o", str(exe), "-L", lib_dir, "-lfitrig", "-Wl,-rpath," + lib_dir], check=True)
    out = subprocess.run([str(exe)], check=True, capture_output=True, text=True).stdout
    assert out.startswith("fitrig-b200")
