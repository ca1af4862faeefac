"""GPU tier, round-2 additions: the entry points and launch modes that had no parity test of their own
("parity-test holes"), and the calls added in round 2.  Same rules as test_parity_gpu.py:
through the C ABI, against the CPU fp64 oracle on the same seeded buffers, tolerances of DESIGN.md section 3.
"""
import ctypes

import numpy as np
import pytest
import torch

import oracle
import paper_2509_21754_b200 as fitrig
import synth
from tests import util
from tests.test_parity_gpu import _check_frequency, check_against_oracle, gpu_run, oracle_delta_at

pytestmark = pytest.mark.gpu
DEV = "cuda:0"


def _collect(ctx, tau, tlisi_out=None, capacity=1 << 16):
    """Everything check_against_oracle looks at, from a context that holds a current map."""
    c, n = ctx.detect(tau, capacity)
    M, mu, sd = ctx.get_stats()
    return {"cands": {tau: (c.copy(), n)}, "M": M, "mu": mu, "sigma": sd, "q": ctx.get_map(0), "tlisi": ctx.get_map(1),
            "raw": ctx.get_raw(), "tlisi_out": tlisi_out, "dims": ctx.map_dims()}


# ------------------------------------------------------------------------------------------
# fitrig_stream from ONE pinned [L, H, W] allocation: every strip travels as one pitched cudaMemcpy2DAsync
# (the path bench.py's e2e number rides), against the per-snapshot copies and against the oracle
# ------------------------------------------------------------------------------------------
@pytest.mark.parametrize("L,H,W,strip,tile", [(6, 300, 252, 64, 32),   # W*4 = 1008: not a multiple of 512; last strip 44 rows
                                              (5, 250, 260, 96, 32),   # partial last tile row inside the last strip
                                              (7, 192, 128, 32, 16),   # many strips, three buffers in rotation
                                              (4, 130, 100, 40, 5)])   # generic time-marching kernel under strips
def test_stream_pitched_copy_equals_per_snapshot_copies_and_oracle(monkeypatch, L, H, W, strip, tile):
    st = synth.gaussian_noise_stack(L, H, W, seed=77, device=DEV)
    st[1:3, H // 3, W // 2] += 40.0
    host = torch.empty((L, H, W), dtype=torch.float32).pin_memory()  # ONE allocation, snapshots equally spaced
    host.copy_(st)
    tau = 2.5
    nstrips = -(-H // strip)
    with fitrig.Context(H, W, L, strip_rows=strip, tile=tile) as ctx:
        U, Ty, Tx = ctx.map_dims()
        h_tl = torch.empty((U, Ty, Tx), dtype=torch.float32).pin_memory()
        ctx.stream([host[s] for s in range(L)], h_tl)
        torch.cuda.synchronize()
        assert ctx.copy_count() == nstrips  # one copy per strip: the pitched path ran
        a = _collect(ctx, tau, h_tl.numpy().copy())
    monkeypatch.setenv("FITRIG_NO_PITCHED_COPY", "1")
    with fitrig.Context(H, W, L, strip_rows=strip, tile=tile) as ctx:
        h_tl2 = torch.empty((U, Ty, Tx), dtype=torch.float32).pin_memory()
        ctx.stream([host[s] for s in range(L)], h_tl2)
        torch.cuda.synchronize()
        assert ctx.copy_count() == nstrips * L
        b = _collect(ctx, tau, h_tl2.numpy().copy())
    assert np.array_equal(a["q"], b["q"]) and np.array_equal(a["tlisi_out"], b["tlisi_out"]) and a["M"] == b["M"]
    for x, y in zip(a["raw"], b["raw"]):
        assert np.array_equal(x, y)
    assert np.array_equal(a["cands"][tau][0], b["cands"][tau][0])
    ref = oracle.run(host.numpy(), tile=tile, tau=tau)
    check_against_oracle(None, a, ref, (tau,), tile, stack_np=host.numpy(), small_tiles=util.needs_slack(H, W, tile))


def test_stream_separately_allocated_snapshots_fall_back_to_per_snapshot_copies():
    st = synth.gaussian_noise_stack(4, 96, 64, seed=3, device=DEV)
    host = [st[s].cpu().pin_memory() for s in range(4)]
    with fitrig.Context(96, 64, 4, strip_rows=32) as ctx:
        ctx.stream(host)
        q = ctx.get_map(0)
        assert ctx.copy_count() in (3, 12)  # 12 unless the allocator happened to space the four buffers equally
    assert np.array_equal(q, gpu_run(st)["q"])


# ------------------------------------------------------------------------------------------
# streams: a side stream, two contexts interleaved on two streams, all entry points chained on one context
# ------------------------------------------------------------------------------------------
def test_stream_from_pageable_host_memory_gives_the_pinned_result():
    """fitrig.h: "pageable memory works, slowly" -- snapshots in ordinary (not page-locked) host memory, as one
    allocation (pitched copies) and as separate numpy arrays, against the pinned run bit for bit; twice on one context."""
    L, H, W, tile = 6, 300, 252, 32
    st = synth.make_stack(synth.scaled(synth.CONFIGS["tiny"], H, W, L=L), device=DEV)[0]
    pinned = gpu_run(st, taus=(3.0,), tile=tile, use_stream=True, strip_rows=64)
    whole = st.cpu()  # pageable, one allocation
    assert not whole.is_pinned()
    separate = [np.array(st[s].cpu().numpy(), copy=True) for s in range(L)]  # pageable, one allocation per snapshot
    with fitrig.Context(H, W, L, tile=tile, strip_rows=64) as ctx:
        U, Ty, Tx = ctx.map_dims()
        h_tl = np.empty((U, Ty, Tx), dtype=np.float32)  # a pageable output too
        for hosts in ([whole[s] for s in range(L)], separate, [whole[s] for s in range(L)]):
            h_tl.fill(-1.0)
            ctx.stream(hosts, h_tl)
            torch.cuda.synchronize()
            c, n = ctx.detect(3.0)
            assert np.array_equal(h_tl, pinned["tlisi_out"]) and np.array_equal(ctx.get_map(0), pinned["q"])
            assert n == pinned["cands"][3.0][1] and np.array_equal(c, pinned["cands"][3.0][0])


@pytest.mark.parametrize("H,W,tile", [(256, 256, 32), (250, 252, 16), (120, 100, 8), (96, 130, 5)])
def test_side_stream_gives_the_default_stream_result(H, W, tile):
    st = synth.make_stack(synth.scaled(synth.CONFIGS["tiny"], H, W), device=DEV)[0]
    ref_run = gpu_run(st, taus=(3.0,), tile=tile)
    side = torch.cuda.Stream()
    with fitrig.Context(H, W, st.shape[0], tile=tile) as ctx:
        U, Ty, Tx = ctx.map_dims()
        d_tl = torch.empty((U, Ty, Tx), dtype=torch.float32, device=DEV)
        side.wait_stream(torch.cuda.current_stream())  # the stack was written on the current stream
        for _ in range(3):  # back to back: the alternating global-maximum keys and the TMA descriptor cache
            ctx.tlisi(st, d_tl, side)
        c, n = ctx.detect(3.0, stream=side)  # synchronises `side`
        host = torch.empty((st.shape[0], H, W), dtype=torch.float32).pin_memory()
        host.copy_(st)
        torch.cuda.synchronize()
        ctx.stream([host[s] for s in range(st.shape[0])], None, side)
        c2, n2 = ctx.detect(3.0, stream=side.cuda_stream)  # a raw stream handle
        q2 = ctx.get_map(0)
    assert np.array_equal(d_tl.cpu().numpy(), ref_run["tlisi"])
    assert np.array_equal(c, ref_run["cands"][3.0][0]) and np.array_equal(c2, c)
    assert np.array_equal(q2, ref_run["q"])


def test_two_contexts_interleaved_on_two_streams():
    a = synth.make_stack(synth.scaled(synth.CONFIGS["tiny"], 256, 256), device=DEV)[0]
    b = synth.gaussian_noise_stack(6, 192, 320, seed=9, device=DEV)
    b[2, 50, 60] += 30.0
    ra, rb = gpu_run(a, taus=(3.0,)), gpu_run(b, taus=(3.0,), tile=16)
    sa, sb = torch.cuda.Stream(), torch.cuda.Stream()
    torch.cuda.synchronize()
    with fitrig.Context(256, 256, 8) as ca, fitrig.Context(192, 320, 6, tile=16) as cb:
        for _ in range(4):
            ca.tlisi(a, None, sa)
            cb.tlisi(b, None, sb)
            ca.detect_launch(3.0, stream=sa)
            cb.detect_launch(3.0, stream=sb)
            outa, outb = (np.zeros(1 << 16, dtype=fitrig.binding.CANDIDATE_DTYPE) for _ in range(2))
            xb, nb, _ = cb.detect_fetch(outb)
            xa, na, _ = ca.detect_fetch(outa)
            assert np.array_equal(xa, ra["cands"][3.0][0]) and np.array_equal(xb, rb["cands"][3.0][0])
        assert np.array_equal(ca.get_map(0), ra["q"]) and np.array_equal(cb.get_map(0), rb["q"])


def test_all_entry_points_chained_on_one_context():
    """fitrig_tlisi -> fitrig_stream -> fitrig_tlisi on ONE context, and a second context that pushes the same
    snapshots: every path must leave the state the next one expects (keys, events, strip buffers, result slots)."""
    st = synth.make_stack(synth.scaled(synth.CONFIGS["tiny"], 160, 192), device=DEV)[0]
    L = st.shape[0]
    host = torch.empty((L, 160, 192), dtype=torch.float32).pin_memory()
    host.copy_(st)
    torch.cuda.synchronize()
    base = gpu_run(st, taus=(3.0,))
    s = torch.cuda.Stream()
    with fitrig.Context(160, 192, L, strip_rows=64) as ctx:
        for rnd in range(3):
            ctx.tlisi(st, None, s)
            c1, _ = ctx.detect(3.0, stream=s)
            ctx.stream([host[i] for i in range(L)], None, s)
            c2, _ = ctx.detect(3.0, stream=s)
            q2 = ctx.get_map(0)
            ctx.tlisi(st)  # default stream right after the side stream
            c3, _ = ctx.detect(3.0)
            assert np.array_equal(c1, base["cands"][3.0][0]) and np.array_equal(c2, c1) and np.array_equal(c3, c1)
            assert np.array_equal(q2, base["q"]) and np.array_equal(ctx.get_map(0), base["q"])
    ref = oracle.run_realtime(st.cpu().numpy(), tile=32, tau=3.0)
    with fitrig.Context(160, 192, 3) as pctx:
        for rnd in range(2):
            got = []
            for snap in [host[i] for i in range(L)] + [None]:
                u, c, n = pctx.push(snap, 3.0, stream=s)
                if u >= 0:
                    got.append((u, pctx.get_map(0)[0].copy()))
            assert [u for u, _ in got] == list(range(L - 2))
            for u, q in got:
                util.assert_map_close(q, ref[u].res.q[0])
            pctx.push_reset()


# ------------------------------------------------------------------------------------------
# fitrig_detect_launch / fitrig_detect_fetch
# ------------------------------------------------------------------------------------------
def test_detect_launch_fetch_pipeline_and_state_errors():
    a = synth.make_stack(synth.scaled(synth.CONFIGS["tiny"], 256, 256), device=DEV)[0]
    b = a.flip(0).contiguous()
    tau, cap = 1.0, 1 << 17  # tiles of 2 pixels at 1 sigma: thousands of candidates
    ra, rb = gpu_run(a, taus=(tau,), tile=2, capacity=cap), gpu_run(b, taus=(tau,), tile=2, capacity=cap)
    outs = [np.zeros(cap, dtype=fitrig.binding.CANDIDATE_DTYPE) for _ in range(2)]
    with fitrig.Context(256, 256, 8, tile=2) as ctx:
        with pytest.raises(fitrig.FitrigError) as e:
            ctx.detect_fetch(outs[0])
        assert e.value.code == fitrig.binding.ERR_STATE
        ctx.tlisi(a)
        ctx.detect_launch(tau, cap)
        ctx.tlisi(b)  # queued behind the first detection: the device never idles
        ctx.detect_launch(tau, cap)
        with pytest.raises(fitrig.FitrigError) as e:
            ctx.detect_launch(tau, cap)  # two in flight
        assert e.value.code == fitrig.binding.ERR_STATE
        with pytest.raises(fitrig.FitrigError) as e:
            ctx.detect(tau)
        assert e.value.code == fitrig.binding.ERR_STATE
        ca, na, _ = ctx.detect_fetch(outs[0])
        cb, nb, _ = ctx.detect_fetch(outs[1])
        assert na == len(ca) and np.array_equal(ca, ra["cands"][tau][0]) and np.array_equal(cb, rb["cands"][tau][0])
        assert na > 4096  # longer than the pinned staging chunk: the rest comes from that slot's device list
        c3, n3 = ctx.detect(tau, cap)
        assert np.array_equal(c3, cb)
        small = np.zeros(10, dtype=fitrig.binding.CANDIDATE_DTYPE)
        ctx.detect_launch(tau, capacity=10)
        cs, ns, _ = ctx.detect_fetch(small)  # FITRIG_ERR_CAPACITY is reported through n_found
        assert ns == nb and np.array_equal(cs, cb[:10])
        # an array shorter than the launch's capacity is refused before the library could write past its end, and a
        # fetch without a buffer fails WITHOUT consuming the launch: the next fetch still delivers it
        ctx.detect_launch(tau, cap)
        with pytest.raises(ValueError):
            ctx.detect_fetch(small)
        n = ctypes.c_int64(0)
        rc = ctx._L.fitrig_detect_fetch(ctx._h, None, ctypes.byref(n), None)
        assert rc == fitrig.binding.ERR_INVALID_ARG and "h_out is NULL" in fitrig.last_error()
        c4, n4, _ = ctx.detect_fetch(outs[0])
        assert n4 == nb and np.array_equal(c4, cb)


# ------------------------------------------------------------------------------------------
# params.batch: B independent stacks per call (BASELINE.json configs[4]: 16 channels, R19), the loop bench.py times
# ------------------------------------------------------------------------------------------
def test_config5_sixteen_channel_batch_reduced_size():
    cfg = synth.scaled(synth.CONFIGS["imgfreq"], 512, 512).replace(n_transients=2, transient_peak=9.0)
    stacks = [synth.make_stack(cfg, device=DEV, channel=ch)[0] for ch in range(cfg.n_channels)]
    B, (L, H, W), tau = len(stacks), stacks[0].shape, 4.0
    assert B == 16
    with fitrig.Context(H, W, L, branch=fitrig.BRANCH_FREQUENCY, batch=B) as ctx:
        U, Ty, Tx = ctx.map_dims()
        d_tl = torch.empty((B, U, Ty, Tx), dtype=torch.float32, device=DEV)
        ctx.tlisi_batch(stacks, d_tl)
        cands, n, per = ctx.detect_batch(tau)
        q, eta, ks = ctx.get_map(0), ctx.get_map(2), ctx.get_map(3).astype(np.int32)
        M, mu, sd = ctx.get_stats()
        tl = ctx.get_map(1)
    assert np.array_equal(d_tl.cpu().numpy(), tl) and per.sum() == n == len(cands) and n > 0
    off = np.concatenate([[0], np.cumsum(per)])
    for b in range(B):
        one = gpu_run(stacks[b], taus=(tau,), branch=fitrig.BRANCH_FREQUENCY)  # the same stack alone: bit-identical
        assert np.array_equal(q[b], one["q"]) and np.array_equal(eta[b], one["eta"]) and np.array_equal(ks[b], one["kstar"])
        assert M[b] == one["M"] and mu[b, 0] == one["mu"][0] and sd[b, 0] == one["sigma"][0]
        assert np.array_equal(cands[off[b]:off[b + 1]], one["cands"][tau][0])
        if b in (0, 7, 15):  # and against the oracle
            ref = oracle.run(stacks[b].cpu().numpy(), tile=32, tau=tau, branch=1)
            g = {"q": q[b], "eta": eta[b], "kstar": ks[b], "mu": mu[b], "sigma": sd[b],
                 "cands": {tau: (cands[off[b]:off[b + 1]], int(per[b]))}}
            _check_frequency(g, ref, (tau,), 32)


@pytest.mark.parametrize("tile,B", [(32, 3), (16, 2), (5, 2), (64, 2), (1, 3), (2, 2), (4, 2)])
def test_image_branch_batch_equals_single_stacks(tile, B):
    stacks = [synth.gaussian_noise_stack(6, 200, 168, seed=40 + b, device=DEV) for b in range(B)]
    for b, s in enumerate(stacks):
        s[1 + b, 20 + 30 * b, 50] += 35.0
    contiguous = torch.stack(stacks).contiguous()
    with fitrig.Context(200, 168, 6, tile=tile, batch=B) as ctx:
        ctx.tlisi(contiguous)  # [B][L][H][W]
        cands, n, per = ctx.detect_batch(2.5)
        q = ctx.get_map(0)
        raw = ctx.get_raw()
        ctx.tlisi_batch(stacks)
        c2, n2 = ctx.detect(2.5)
        assert np.array_equal(c2, cands) and np.array_equal(ctx.get_map(0), q)
        with pytest.raises(fitrig.FitrigError):
            ctx.stream([torch.zeros(200, 168).pin_memory()] * 6)
    off = np.concatenate([[0], np.cumsum(per)])
    for b in range(B):
        one = gpu_run(stacks[b], taus=(2.5,), tile=tile)
        assert np.array_equal(q[b], one["q"]) and np.array_equal(cands[off[b]:off[b + 1]], one["cands"][2.5][0])
        for x, y in zip(raw, one["raw"]):
            assert np.array_equal(x[b], y)
    with pytest.raises(fitrig.FitrigError) as e:
        fitrig.Context(64, 64, 4, batch=2, row_offset=32)
    assert e.value.code == fitrig.binding.ERR_INVALID_ARG


@pytest.mark.parametrize("tile,H,W", [(32, 64, 96), (8, 40, 64), (5, 40, 50)])
def test_back_to_back_batch_calls_without_detect(tile, H, W):
    """A caller that only consumes d_tlisi: call after call on a batch context, nothing in between.  The kernels of
    stacks b >= 1 do not wait at their start, so they must not become schedulable before the previous call's finalise
    (which still reads the records and resets the maximum keys) has completed.  Small images, so that the grids of
    consecutive kernels fit on the device together."""
    B, L = 3, 5
    first = [synth.gaussian_noise_stack(L, H, W, seed=60 + b, device=DEV) for b in range(B)]
    second = [(2.0 + b) * synth.gaussian_noise_stack(L, H, W, seed=70 + b, device=DEV) for b in range(B)]  # other maxima
    for b in range(B):
        second[b][1, 3 + b, 7] += 90.0 + 10.0 * b
    exp = []
    for stacks in (first, second):
        runs = [gpu_run(s, taus=(3.0,), tile=tile) for s in stacks]
        exp.append((torch.from_numpy(np.stack([r["tlisi"] for r in runs])).to(DEV), np.array([r["M"] for r in runs])))
    assert not np.array_equal(exp[0][1], exp[1][1])
    with fitrig.Context(H, W, L, tile=tile, batch=B) as ctx:
        U, Ty, Tx = ctx.map_dims()
        outs = [torch.empty((B, U, Ty, Tx), dtype=torch.float32, device=DEV) for _ in range(2)]
        for it in range(25):
            outs[0].fill_(-1.0)
            outs[1].fill_(-1.0)
            ctx.tlisi_batch(first, outs[0])
            ctx.tlisi_batch(second, outs[1])
            if it % 2:  # and a third call straight behind the second
                ctx.tlisi_batch(first, outs[0])
            torch.cuda.synchronize()
            assert torch.equal(outs[0], exp[0][0]) and torch.equal(outs[1], exp[1][0]), it
            M, _, _ = ctx.get_stats()
            assert np.array_equal(M, exp[it % 2 == 0][1]), it


@pytest.mark.parametrize("tile", [1, 2])
def test_frequency_branch_batch_of_pixel_tiles_equals_single_stacks(tile):
    # per-pixel detection keeps 8-byte records: stacks b >= 1 of a batch must land at their own rows
    B, L, H, W, tau = 3, 10, 72, 88, 3.0
    cfg = synth.scaled(synth.CONFIGS["imgfreq"], H, W, L=L).replace(n_transients=2, transient_peak=14.0, period=4)
    stacks = [synth.make_stack(cfg, device=DEV, channel=ch)[0] for ch in range(B)]
    with fitrig.Context(H, W, L, tile=tile, branch=fitrig.BRANCH_FREQUENCY, batch=B) as ctx:
        ctx.tlisi_batch(stacks)
        cands, n, per = ctx.detect_batch(tau)
        q, eta, ks = ctx.get_map(0), ctx.get_map(2), ctx.get_map(3).astype(np.int32)
        M, mu, sd = ctx.get_stats()
    off = np.concatenate([[0], np.cumsum(per)])
    for b in range(B):
        one = gpu_run(stacks[b], taus=(tau,), tile=tile, branch=fitrig.BRANCH_FREQUENCY)
        assert np.array_equal(q[b], one["q"]) and np.array_equal(eta[b], one["eta"]) and np.array_equal(ks[b], one["kstar"])
        assert M[b] == one["M"] and mu[b, 0] == one["mu"][0] and sd[b, 0] == one["sigma"][0]
        assert np.array_equal(cands[off[b]:off[b + 1]], one["cands"][tau][0])
    # the last stack against the oracle: q within 1e-4 + the derived fp32 input-rounding bound of tiles of a few pixels
    # (util.fp32_slack, as in check_against_oracle), eta within what that moves a DFT magnitude by (util.eta_bound's argument)
    snaps = stacks[B - 1].cpu().numpy()
    ref = oracle.run(snaps, tile=tile, tau=tau, branch=1)
    res = ref.res
    eS, eM, eR = util.fp32_slack(snaps, tile)
    prod = res.sumD * res.maxD * res.sumR
    slack = ((res.sumD + eS) * (res.maxD + eM) * (np.abs(res.sumR) + eR) - prod) * np.abs(res.q / np.where(prod == 0, 1.0, prod))
    util.assert_map_close(q[B - 1], res.q, slack=slack)
    bound = 2.0 * (util.Q_RTOL * np.abs(res.q) + slack).sum(axis=0)
    assert np.all(np.abs(eta[B - 1] - ref.eta) <= bound + 2e-7 * np.abs(ref.eta))


# ------------------------------------------------------------------------------------------
# real-time form of the image-frequency branch (R29): fitrig_push on a frequency-branch context
# ------------------------------------------------------------------------------------------
@pytest.mark.parametrize("H,W,tile,window,harmonics", [(128, 160, 16, 8, 1), (96, 96, 8, 5, 1), (128, 128, 32, 12, 2),
                                                        (90, 100, 12, 6, 1)])
def test_push_frequency_branch_matches_oracle(H, W, tile, window, harmonics):
    cfg = synth.scaled(synth.CONFIGS["imgfreq"], H, W, L=16).replace(n_transients=2, transient_peak=14.0, period=4)
    st, _ = synth.make_stack(cfg, device=DEV)
    st[6, 7, 9] = 300.0  # the running maximum jumps in the middle
    L, tau, Uw = st.shape[0], 2.0, window - 2
    ref = oracle.run_realtime_frequency(st.cpu().numpy(), window, tile=tile, tau=tau, harmonics=harmonics)
    host = [st[s].cpu().pin_memory() for s in range(L)]
    with fitrig.Context(H, W, window, tile=tile, branch=fitrig.BRANCH_FREQUENCY, harmonics=harmonics) as ctx:
        U, Ty, Tx = ctx.map_dims()
        assert U == Uw
        d_tl = torch.empty((Ty, Tx), dtype=torch.float32, device=DEV)
        seen = 0
        for snap in host + [None]:
            u, c, n = ctx.push(snap, tau, d_tl)
            if u < 0:
                continue
            assert u == seen
            seen += 1
            if ref[u] is None:
                assert n == 0
                continue
            r = ref[u]
            M, mu, sd = ctx.get_stats()
            assert M == np.float32(r.res.M)
            cube = ctx.get_map(0)  # ring: map row (n mod U) holds unit n
            order = [(u - Uw + 1 + j) % Uw for j in range(Uw)]
            util.assert_map_close(cube[order], r.res.q)
            assert np.allclose(d_tl.cpu().numpy(), 1.0 - cube[u % Uw], atol=1e-6)
            g = {"q": cube[order], "eta": ctx.get_map(2), "kstar": ctx.get_map(3).astype(np.int32), "mu": mu, "sigma": sd,
                 "cands": {tau: (c.copy(), n)}}
            small = util.needs_slack(H, W, tile)
            bound = util.eta_bound(r.res.q, harmonics, eps_q=util.Q_RTOL if (small or tile != 32) else util.EPS_Q_FP32)
            assert np.all(np.abs(g["eta"] - r.eta) <= bound + 2e-7 * np.abs(r.eta))
            band = util.eta_z_band(r.eta, r.z, r.sigma[0], bound)
            lst = [(int(k["x"]), int(k["y"]), int(k["snapshot"]), float(k["score"]),
                    (int(k["y"]) // tile) * Tx + int(k["x"]) // tile, 0) for k in c]
            util.compare_candidates(lst, r.z[None], r.mu, r.sigma, tau, Tx, Ty * Tx, band=band[None])
        assert seen == L - 2
        # a second pass after a reset reproduces the last result bit for bit
        last = (c.copy(), ctx.get_map(2).copy())
        ctx.push_reset()
        for snap in host + [None]:
            u, c, n = ctx.push(snap, tau)
        assert np.array_equal(c, last[0]) and np.array_equal(ctx.get_map(2), last[1])


@pytest.mark.parametrize("tile", [1, 2, 4])
def test_push_frequency_branch_small_tiles_fill_their_own_ring_rows(tile):
    """Tiles of one pixel keep 8-byte records: ring row n mod U of the cube must land where the finalise, the spectrum
    and the getters read it.  The cube after the last push is the map of the last window of snapshots under the running
    maximum, so it is compared bit for bit with a resident run on those snapshots with M_override = that maximum."""
    H, W, window, L, tau = 40, 48, 6, 12, 2.0
    cfg = synth.scaled(synth.CONFIGS["imgfreq"], H, W, L=L).replace(n_transients=2, transient_peak=14.0, period=4)
    st, _ = synth.make_stack(cfg, device=DEV)
    st[3, 7, 9] = 300.0  # the running maximum comes from a snapshot that has left the window
    Uw = window - 2
    host = [st[s].cpu().pin_memory() for s in range(L)]
    with fitrig.Context(H, W, window, tile=tile, branch=fitrig.BRANCH_FREQUENCY) as ctx:
        for snap in host + [None]:
            u, c, n = ctx.push(snap, tau)
        M, mu, sd = ctx.get_stats()
        cube, eta, ks = ctx.get_map(0), ctx.get_map(2), ctx.get_map(3).astype(np.int32)
        c = c.copy()
    assert u == L - 3 and M == np.float32(300.0)
    order = [(u - Uw + 1 + j) % Uw for j in range(Uw)]
    one = gpu_run(st[L - window:].contiguous(), taus=(tau,), tile=tile, branch=fitrig.BRANCH_FREQUENCY, M_override=300.0)
    assert np.array_equal(cube[order], one["q"])
    # |F_k| does not depend on where the ring starts, up to the rounding of the fp64 sums (and one fp32 rounding of eta)
    np.testing.assert_allclose(eta, one["eta"], rtol=1e-6, atol=0)
    ref = oracle.run(st[L - window:].cpu().numpy(), tile=tile, tau=tau, branch=1, M=300.0)
    slack = None
    if util.needs_slack(H, W, tile):  # the derived fp32 input-rounding bound, as in check_against_oracle
        res = ref.res
        eS, eM, eR = util.fp32_slack(st[L - window:].cpu().numpy(), tile)
        prod = res.sumD * res.maxD * res.sumR
        slack = ((res.sumD + eS) * (res.maxD + eM) * (np.abs(res.sumR) + eR) - prod) * np.abs(res.q / np.where(prod == 0, 1.0, prod))
    util.assert_map_close(cube[order], ref.res.q, slack=slack)
    sure = np.abs(one["eta"] - (one["mu"][0] + tau * one["sigma"][0])) > 1e-5 * np.abs(one["eta"])  # away from the threshold
    got = {(int(k["x"]), int(k["y"])) for k in c}
    exp = {(int(k["x"]), int(k["y"])) for k in one["cands"][tau][0]}
    Tx = one["dims"][2]
    for (x, y) in got ^ exp:
        assert not sure[y // tile, x // tile]
    assert len(got & exp) > 0


# ------------------------------------------------------------------------------------------
# row shards: frequency branch (second exchange), constant maps, strips that end inside a 32-row block
# ------------------------------------------------------------------------------------------
@pytest.mark.parametrize("H,W,world", [(256, 256, 2), (250, 252, 3)])
def test_row_shards_frequency_branch_reproduce_the_whole_image(H, W, world):
    from paper_2509_21754_b200 import shard
    cfg = synth.scaled(synth.CONFIGS["imgfreq"], H, W, L=12).replace(n_transients=2, transient_peak=12.0, period=4)
    st, _ = synth.make_stack(cfg, device=DEV)
    L, tau, tile = cfg.L, 1.5, 16
    whole = gpu_run(st, taus=(tau,), tile=tile, branch=fitrig.BRANCH_FREQUENCY)
    rows = shard.row_shards(H, tile, world)
    ctxs, vecs, evs = [], [], []
    try:
        for (r0, r1) in rows:
            ctx = fitrig.Context(r1 - r0, W, L, row_offset=r0, tile=tile, branch=fitrig.BRANCH_FREQUENCY)
            ctxs.append(ctx)
            ctx.tlisi(st[:, r0:r1].contiguous())
            v = torch.empty(2 + 2 * (L - 2), dtype=torch.float64, device=DEV)
            ctx.shard_export(v)
            vecs.append(v)
        allv = torch.stack(vecs).contiguous()
        for ctx in ctxs:  # first exchange: M, and mu / sigma of q
            ctx.shard_import(allv, world)
            e = torch.empty(3, dtype=torch.float64, device=DEV)
            ctx.shard_export_eta(e)
            evs.append(e)
        alle = torch.stack(evs).contiguous()
        etas, lists = [], []
        for ctx, (r0, r1) in zip(ctxs, rows):  # second exchange: mean and std of eta over the whole image
            ctx.shard_import_eta(alle, world)
            c, n = ctx.detect(tau)
            M, mu, sd = ctx.get_stats()
            assert M == whole["M"]
            assert abs(mu[0] - whole["mu"][0]) <= 1e-9 * abs(whole["mu"][0]) and abs(sd[0] - whole["sigma"][0]) <= 1e-7 * whole["sigma"][0]
            etas.append(ctx.get_map(2))
            lists.append(c.copy())
            assert all(r0 <= int(y) < r1 for y in c["y"])
    finally:
        for ctx in ctxs:
            ctx.close()
    assert np.array_equal(np.concatenate(etas, axis=0), whole["eta"])  # same q, same fp64 DFT
    merged = np.concatenate(lists)  # one row of the map per shard, shards in row order
    ref_c, ref_n = whole["cands"][tau]
    keep = lambda c: {(int(r["snapshot"]), int(r["y"]), int(r["x"])) for r in c if abs(float(r["score"]) - tau) > 1e-5}
    assert keep(merged) == keep(ref_c) and ref_n > 0


@pytest.mark.parametrize("branch,H,W,tile,world", [(0, 250, 252, 32, 3), (1, 256, 256, 16, 2), (0, 96, 128, 1, 2)])
def test_row_shards_streamed_from_whole_host_snapshots(branch, H, W, tile, world):
    """ShardedContext.stream / shard_host_rows (SURVEY.md 8(e), config 4 over several GPUs): every shard copies only its
    own rows of the whole pinned snapshots through fitrig_stream.  One GPU here, so the shards run one after another and
    the all-gather is the stack of their export vectors; a world of one goes through ShardedContext.stream itself."""
    from paper_2509_21754_b200 import shard
    L, tau = (12, 2.0) if branch else (8, 3.0)
    cfg = synth.scaled(synth.CONFIGS["imgfreq" if branch else "tiny"], H, W, L=L)
    st = synth.make_stack(cfg, device=DEV)[0]
    host = st.cpu().pin_memory()
    snaps = [host[s] for s in range(L)]
    whole = gpu_run(st, taus=(tau,), tile=tile, branch=branch, capacity=1 << 18)
    with shard.ShardedContext(H, W, L, 0, 1, tile=tile, branch=branch) as sc:  # world = 1: no process group needed
        U, Ty, Tx = sc.ctx.map_dims()
        d_tl = torch.empty((U, Ty, Tx), dtype=torch.float32, device=DEV)
        sc.stream(snaps, d_tl, torch.cuda.Stream(device=DEV))
        torch.cuda.synchronize()
        c1, n1 = sc.detect(tau, 1 << 18)
        assert np.array_equal(sc.ctx.get_map(0), whole["q"]) and np.array_equal(d_tl.cpu().numpy(), whole["tlisi"])
        assert n1 == whole["cands"][tau][1] or abs(n1 - whole["cands"][tau][1]) <= 2  # (z from sums of p: last bits)
    rows = shard.row_shards(H, tile, world)
    ctxs, vecs, qs = [], [], []
    try:
        for (r0, r1) in rows:
            ctx = fitrig.Context(r1 - r0, W, L, row_offset=r0, tile=tile, branch=branch)
            ctxs.append(ctx)
            ctx.stream(shard.shard_host_rows(snaps, r0, r1))
            v = torch.empty(2 + 2 * (L - 2), dtype=torch.float64, device=DEV)
            ctx.shard_export(v)
            vecs.append(v)
        allv = torch.stack(vecs).contiguous()
        for ctx in ctxs:
            ctx.shard_import(allv, world)
            qs.append(ctx.get_map(0))
            assert ctx.get_stats()[0] == whole["M"]
        assert sum(c.copy_count() for c in ctxs) > 0
    finally:
        for ctx in ctxs:
            ctx.close()
    assert np.array_equal(np.concatenate(qs, axis=1), whole["q"])


def test_row_shards_of_a_constant_map_have_zero_sigma_and_no_candidates():
    """a one-pass variance of the shards' sums could turn sigma == 0 (R4) into a tiny positive number and
    spurious large z.  Every tile of this stack has the same raw sums, so q is constant over the image."""
    tile, L, world = 32, 5, 3
    one = synth.gaussian_noise_stack(L, tile, tile, seed=5, device=DEV)
    st = one.repeat(1, 6, 4).contiguous()  # 6 x 4 identical tiles
    H, W = st.shape[1:]
    from paper_2509_21754_b200 import shard
    rows = shard.row_shards(H, tile, world)
    ctxs, vecs = [], []
    try:
        for (r0, r1) in rows:
            ctx = fitrig.Context(r1 - r0, W, L, row_offset=r0)
            ctxs.append(ctx)
            ctx.tlisi(st[:, r0:r1].contiguous())
            v = torch.empty(2 + 2 * (L - 2), dtype=torch.float64, device=DEV)
            ctx.shard_export(v)
            vecs.append(v)
        allv = torch.stack(vecs).contiguous()
        for ctx in ctxs:
            ctx.shard_import(allv, world)
            M, mu, sd = ctx.get_stats()
            assert np.all(sd == 0.0) and np.all(mu > 0)
            assert ctx.detect(0.0)[1] == 0
    finally:
        for ctx in ctxs:
            ctx.close()
    whole = gpu_run(st, taus=(0.0,))
    assert np.all(whole["sigma"] == 0.0) and whole["cands"][0.0][1] == 0


@pytest.mark.parametrize("tile,strip", [(16, 48), (8, 40), (4, 20), (1, 33), (2, 50)])
def test_strips_that_end_inside_a_32_row_block(tile, strip):
    """a strip whose height is not a multiple of 32 shares its last 32-row block with the next strip; the
    cells of that overhang belong to the next strip and must be neither written nor re-read by this one."""
    st = synth.gaussian_noise_stack(5, 200, 128, seed=21, device=DEV)
    a = gpu_run(st, taus=(2.5,), tile=tile)
    b = gpu_run(st, taus=(2.5,), tile=tile, use_stream=True, strip_rows=strip)
    assert np.array_equal(a["raw"][1], b["raw"][1]) and np.array_equal(a["raw"][3], b["raw"][3])  # max and arg-max exact
    np.testing.assert_allclose(b["q"], a["q"], rtol=2e-6)  # (strips off the 32-row grid take the generic kernel: other sum order)
    ref = oracle.run(st.cpu().numpy(), tile=tile, tau=2.5)
    check_against_oracle(st, b, ref, (2.5,), tile, small_tiles=util.needs_slack(200, 128, tile))


def test_more_units_than_a_grid_dimension():
    """U > 65535 used to overflow gridDim.y of the finalise kernel."""
    L = 66000
    st = synth.gaussian_noise_stack(L, 32, 64, seed=8, device=DEV)
    g = gpu_run(st, taus=(0.5,), capacity=1 << 18)
    assert g["dims"] == (L - 2, 1, 2)
    ref = oracle.run(st.cpu().numpy(), tile=32, tau=0.5)
    util.assert_map_close(g["q"], ref.res.q)
    assert g["cands"][0.5][1] == ref.cands.n_found  # two tiles per unit: z = +-1, one candidate per unit
    with pytest.raises(fitrig.FitrigError) as e:
        fitrig.Context(32, 32, 9000, branch=fitrig.BRANCH_FREQUENCY)  # the DFT's twiddle table has a stated limit
    assert e.value.code == fitrig.binding.ERR_INVALID_ARG


# ------------------------------------------------------------------------------------------
# fitrig_localise: sub-tile localisation by interpolating eta (R28) against oracle.localise
# ------------------------------------------------------------------------------------------
METHODS = [fitrig.INTERP_BILINEAR, fitrig.INTERP_BICUBIC, fitrig.INTERP_SPLINE, fitrig.INTERP_MAKIMA]


def _centre_candidates(Ty, Tx, tile, tiles):
    c = np.zeros(len(tiles), dtype=fitrig.binding.CANDIDATE_DTYPE)
    for k, t in enumerate(tiles):
        ty, tx = divmod(int(t), Tx)
        c[k] = (tx * tile + tile // 2, ty * tile + tile // 2, 1, 0.0)
    return c


def _check_positions(pos, eta64, tile, tiles, method, r, slack):
    """The position is an arg-max over a lattice: unique up to values that agree within `slack` (R23's rule for
    integer decisions taken on floating-point values): wherever the library's lattice point differs from the oracle's,
    the ORACLE's surface there must be within slack of the oracle's maximum, and it must lie on the lattice."""
    ref = oracle.localise(eta64, tile, tiles, method, r)
    Ty, Tx = eta64.shape
    same = (pos["x"] == ref.x) & (pos["y"] == ref.y)
    for k in np.argwhere(~same).reshape(-1):
        u, v = (pos["x"][k] + 0.5) / tile - 0.5, (pos["y"][k] + 0.5) / tile - 0.5
        ty, tx = divmod(int(tiles[k]), Tx)
        assert abs(u - tx) <= 1 + 1e-12 and abs(v - ty) <= 1 + 1e-12 and 0 <= u <= Tx - 1 and 0 <= v <= Ty - 1
        du, dv = (u - tx) * tile * r, (v - ty) * tile * r
        assert abs(du - round(du)) < 1e-9 and abs(dv - round(dv)) < 1e-9  # a lattice point
        assert oracle.interp_eval(eta64, method, u, v)[0] >= ref.value[k] - slack[k]
    assert np.all(np.abs(pos["value"] - ref.value) <= slack + 1e-12 * np.abs(ref.value))
    return int(same.sum())


@pytest.mark.parametrize("method", METHODS)
@pytest.mark.parametrize("Ty,Tx,tile,r", [(6, 7, 8, 1), (12, 9, 4, 3), (3, 3, 8, 2), (2, 5, 5, 1), (1, 4, 8, 2), (4, 1, 4, 1),
                                          (1, 1, 8, 1), (40, 33, 4, 1), (5, 6, 32, 1)])
def test_localise_supplied_surface_matches_oracle(method, Ty, Tx, tile, r):
    rng = np.random.default_rng(100 * Ty + Tx + method)
    eta = rng.normal(size=(Ty, Tx)).astype(np.float32)
    eta[Ty // 2, Tx // 2] += 5.0
    if Ty > 2 and Tx > 3:
        eta[1, 2] = eta[1, 3] = 7.0  # a source shared by two tiles: a plateau / a symmetric peak between the centres
    tiles = list(range(Ty * Tx)) if Ty * Tx <= 60 else list(rng.choice(Ty * Tx, 40, replace=False))
    cands = _centre_candidates(Ty, Tx, tile, tiles)
    with fitrig.Context(Ty * tile, Tx * tile, 4, tile=tile, branch=fitrig.BRANCH_FREQUENCY) as ctx:
        pos = ctx.localise(cands, method, r, eta=eta)
    # the same fp32 matrix widened exactly; both sides compute in fp64: only the rounding order differs
    same = _check_positions(pos, eta.astype(np.float64), tile, tiles, method, r, np.full(len(tiles), 1e-11))
    assert same >= 0.95 * len(tiles)


@pytest.mark.parametrize("method", [fitrig.INTERP_BICUBIC, fitrig.INTERP_SPLINE])
def test_localise_paraboloid_peak(method):
    tile, Ty, Tx = 32, 7, 9
    u0, v0 = 4.3, 2.6
    U, V = np.meshgrid(np.arange(Tx, dtype=np.float64), np.arange(Ty, dtype=np.float64))
    eta = (10.0 - (U - u0) ** 2 - (V - v0) ** 2).astype(np.float32)
    x0, y0 = (u0 + 0.5) * tile - 0.5, (v0 + 0.5) * tile - 0.5
    with fitrig.Context(Ty * tile, Tx * tile, 4, branch=fitrig.BRANCH_FREQUENCY) as ctx:
        for r in (1, 4):
            pos = ctx.localise(_centre_candidates(Ty, Tx, tile, [3 * Tx + 4, 2 * Tx + 4, 3 * Tx + 5]), method, r, eta=eta)
            for k in range(3):  # the lattices of the three tiles differ by whole tiles: the same nearest point
                assert abs(pos["x"][k] - x0) <= 0.5 / r + 1e-4 and abs(pos["y"][k] - y0) <= 0.5 / r + 1e-4


def test_localise_after_detect_on_reduced_config5():
    cfg = synth.scaled(synth.CONFIGS["imgfreq"], 1024, 1024).replace(n_transients=3, transient_peak=9.0)
    st, truth = synth.make_stack(cfg, device=DEV)
    tau = 5.0
    with fitrig.Context(1024, 1024, cfg.L, branch=fitrig.BRANCH_FREQUENCY) as ctx:
        with pytest.raises(fitrig.FitrigError) as e:
            ctx.localise(_centre_candidates(32, 32, 32, [5]), fitrig.INTERP_SPLINE)
        assert e.value.code == fitrig.binding.ERR_STATE  # no eta yet
        ctx.tlisi(st)
        cands, n = ctx.detect(tau)
        assert n > 0
        got = {m: ctx.localise(cands, m, 2) for m in METHODS}
        with pytest.raises(fitrig.FitrigError) as e:
            ctx.localise(cands, 7)
        assert e.value.code == fitrig.binding.ERR_INVALID_ARG
    ref = oracle.run(st.cpu().numpy(), tile=32, tau=tau, branch=1)
    Tx = ref.res.Tx
    tiles = [(int(c["y"]) // 32) * Tx + int(c["x"]) // 32 for c in cands]
    # the surface is a combination of eta values with weights whose absolute sum is at most 1.25^2 (Keys), about 2.4
    # (spline) per point: what eta's bound (util.eta_bound) can move a surface value by, both ways
    bound = util.eta_bound(ref.res.q)
    slack = np.full(len(tiles), 2 * 2.5 * float(bound.max()) + 1e-6 * float(np.abs(ref.eta).max()))
    for m in METHODS:
        _check_positions(got[m], ref.eta, 32, tiles, m, 2, slack)
    hit = 0
    for t in truth.transients:  # a localised transient lies within its tile's reach
        for k, c in enumerate(cands):
            if int(c["x"]) // 32 == t.x // 32 and int(c["y"]) // 32 == t.y // 32:
                hit += 1
                assert abs(got[fitrig.INTERP_SPLINE]["x"][k] - t.x) <= 32 and abs(got[fitrig.INTERP_SPLINE]["y"][k] - t.y) <= 32
    assert hit > 0
    with fitrig.Context(256, 256, 8) as ctx:  # image branch
        ctx.tlisi(st[:8, :256, :256].contiguous())
        with pytest.raises(fitrig.FitrigError) as e:
            ctx.localise(_centre_candidates(8, 8, 32, [3]), fitrig.INTERP_SPLINE)
        assert e.value.code == fitrig.binding.ERR_INVALID_ARG
