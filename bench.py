#!/usr/bin/env python
"""bench.py -- the SU(3)xSU(3) streaming benchmark (BASELINE.json metric) on N B200s.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--L 64] [--impl ours|reference]
    python -m torch.distributed.run --nnodes=1 --nproc-per-node N ... bench.py --gpus N ...

A STEP is one pass of the whole hot path over one batch of
seeded synthetic SU(3) fields on an L^4 lattice (default L = 64, fp64: the HBM-bound top of the
volume sweep, BASELINE.json configs[4]; Listing 3):

    A5  convert  x, y, w : scalar -> vector (W=4)          3 launches, 2 field streams each
    A1  mul      zs = xs*ys          (scalar layout)       3 streams, 198 flop/matrix
    A2  mul      zv = xv*yv          (vector layout W=4)   3 streams
    A3  mul3     z3 = xv*yv*wv       (vector layout)       4 streams, 396 flop/matrix
    A4  mul_add  z4 = xs*ys + vs     (scalar layout)       4 streams, 216 flop/matrix
    A5  convert  zb = scalar(zv)                           2 streams
    A6  copy     zc = zs             (the ceiling kernel)  2 streams

`value` = algorithmic bytes of the step (S9: 24 field streams) / device time, inputs resident in HBM.
`e2e`   = the same step with HOST buffers: x, y, w, v come from pinned host memory (x, y and the A1
          result through the C-ABI call su3_mul_host) and the four results go back to the host,
          all inside the timed region.
One JSON line on stdout (rank 0); progress goes to stderr.
"""
import argparse
import json
import os
import subprocess
import sys
import tempfile
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

import numpy as np

METRIC = "su3xsu3_stream_GBps"
UNIT = "GB/s"
FLOPS = {"mul": 198, "mul3": 396, "mul_add": 216, "convert": 0, "copy": 0, "add": 18}
STREAMS = {"mul": 3, "mul3": 4, "mul_add": 4, "convert": 2, "copy": 2, "add": 3}
E2E_CHUNKS = int(os.environ.get("SU3_E2E_CHUNKS", "16"))  # chunks of the host pipelines in the e2e leg
W64, W32 = 4, 8  # vector lengths of the configs: fp64 W=4, fp32 W=8 (64-byte element vectors)


def log(*a):
    print(*a, file=sys.stderr, flush=True)


def parse_args():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=20)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--L", type=int, default=64, help="local lattice extent per GPU (L^4 sites)")
    ap.add_argument("--impl", choices=["ours", "reference"], default="ours")
    ap.add_argument("--no-sweep", action="store_true", help="skip the volume sweep (configs[4]) after the timed steps")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--no-cpu", action="store_true", help="skip the cpu_baseline leg")
    ap.add_argument("--profile-pass", action="store_true",
                    help="launch every kernel variant of the library once at 48^4 (no timing): the command ncu wraps "
                         "for profiles/*_all_kernels.md")
    ap.add_argument("--cpu-L", type=int, default=32, help="lattice extent of the oracle's bounded sample")
    return ap.parse_args()


def measured_peak():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    try:
        with open(p) as f:
            return float(json.load(f)["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)"
    except Exception:
        return 6650.0, "fallback (B200_PROFILING.md: 6.65 TB/s)"


# ---------------------------------------------------------------------------- the oracle legs
def oracle_step(L, reps, threads=None):
    """Time the oracle, as it stands, on `reps` passes of one step (rows A1-A6; A6 is a memcpy) of an L^4
    fp64 lattice.  Returns (seconds per pass [reps], bytes a pass moves by S9's accounting, threads used)."""
    import oracle
    import su3gen
    if threads:
        oracle.set_num_threads(threads)
    seed = su3gen.config_seed(5)
    gs, gv = oracle.Geom(L), oracle.Geom(L, layout=oracle.su3_oracle.VECTOR, W=W64)
    n = gs.nmat
    xs, ys, ws = (su3gen.su3_field(seed, f, n).view(np.float64).reshape(-1) for f in (0, 1, 2))
    vs = su3gen.gaussian_field(seed, 3, n).view(np.float64).reshape(-1)
    times = []
    for _ in range(reps):
        t0 = time.perf_counter()
        xv, yv, wv = (oracle.convert(gv, gs, a) for a in (xs, ys, ws))
        zs = oracle.mul(gs, xs, ys)
        zv = oracle.mul(gv, xv, yv)
        z3 = oracle.mul3(gv, xv, yv, wv)
        z4 = oracle.mul_add(gs, xs, ys, vs)
        zb = oracle.convert(gs, gv, zv)
        zc = zs.copy()
        times.append(time.perf_counter() - t0)
    assert np.array_equal(zb, zs) and zc.size == zs.size and z3.size == z4.size
    return times, 24 * n * 144, oracle.num_threads()


def run_reference(args, rank):
    """--impl reference: the oracle on the host cores, same metric/config; every step is one pass over a
    bounded sample (a smaller lattice of the same sweep) so that W+K passes end within a few minutes."""
    if rank != 0:
        return
    L = min(args.cpu_L, args.L)
    if args.warmup + args.steps > 30:
        L = min(L, 24)
    times, nbytes, threads = oracle_step(L, args.warmup + args.steps)
    timed = times[args.warmup:]
    sec = sum(timed) / len(timed)
    val = nbytes / sec / 1e9
    sample = "every step = rows A1-A6 on a %d^4 fp64 lattice (a smaller point of the same sweep; workload %d^4)" % (L, args.L)
    print(json.dumps({
        "impl": "reference", "metric": METRIC, "value": val, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": sec * 1e3, "higher_is_better": True, "scaling": "weak",
        "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {"workload": "cfg5 volume sweep top: %d^4 fp64, rows A1-A6" % args.L, "sample_L": L},
        "cpu_baseline": {"value": val, "unit": UNIT, "cores": threads, "kind": "oracle", "sample": sample},
        "e2e": {"value": val, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
    }), flush=True)


# ---------------------------------------------------------------------------- clocks during the timed region
CLOCK_Q = ("index,clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.active,clocks_event_reasons.hw_slowdown,"
           "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
           "clocks_event_reasons.sw_power_cap")


class ClockSampler:
    def __init__(self, gpu_index):
        self.f = tempfile.NamedTemporaryFile("w+", suffix=".csv", delete=False)
        self.p = None
        try:
            self.p = subprocess.Popen(["nvidia-smi", "-i", str(gpu_index), "--query-gpu=" + CLOCK_Q,
                                       "--format=csv,noheader,nounits", "-lms", "100"],
                                      stdout=self.f, stderr=subprocess.DEVNULL)
        except OSError:
            pass

    def stop(self):
        if self.p is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        time.sleep(0.15)
        self.p.terminate()
        try:
            self.p.wait(timeout=5)
        except subprocess.TimeoutExpired:
            self.p.kill()
        self.f.flush()
        self.f.seek(0)
        sm, smax, reasons, power = [], [], set(), []
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for line in self.f:
            c = [t.strip() for t in line.split(",")]
            if len(c) < 9:
                continue
            try:
                sm.append(float(c[1])); smax.append(float(c[2])); power.append(float(c[3]))
            except ValueError:
                continue
            for nm, v in zip(names, c[5:9]):
                if v.lower().startswith("active"):
                    reasons.add(nm)
        self.f.close()
        os.unlink(self.f.name)
        if not sm:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["no samples"]}
        return {"sm_mhz": float(np.median(sm)), "sm_max_mhz": max(smax), "power_w_max": max(power),
                "samples": len(sm), "reasons": sorted(reasons)}


# ---------------------------------------------------------------------------- our arm
def run_ours(args, rank, world, local_rank):
    import torch

    import paper_1710_09409_b200 as su3   # raises if libsu3stream.so cannot be built/loaded: no fallback
    import su3gen
    from paper_1710_09409_b200 import shard

    if not torch.cuda.is_available():
        raise RuntimeError("bench.py needs a CUDA device; there is no CPU fallback (use --impl reference for the oracle)")
    ngpu = torch.cuda.device_count()
    dev = torch.device("cuda", local_rank % ngpu)
    torch.cuda.set_device(dev)
    dist = None
    coll_dev = dev
    if world > 1:
        import torch.distributed as dist
        if ngpu >= world:
            dist.init_process_group("nccl", device_id=dev)
        else:
            # fewer GPUs than ranks (a functional check of the N > 1 path only): ranks share GPUs, plumbing over gloo.
            # No kernel of one rank ever waits for another rank, so sharing a GPU cannot deadlock.
            log("[rank %d] %d GPU(s) for %d ranks: sharing devices, gloo plumbing -- NOT a scaling measurement" % (rank, ngpu, world))
            dist.init_process_group("gloo")
            coll_dev = torch.device("cpu")

    def barrier():
        if dist is not None:
            dist.barrier()
        torch.cuda.synchronize()

    L = args.L
    info = su3.su3_device_info()
    F64, F32, SC, VE = su3.SU3_F64, su3.SU3_F32, su3.SU3_SCALAR, su3.SU3_VECTOR
    ds, dv = su3.make_desc(L), su3.make_desc(L, layout=VE, W=W64)
    nmat = L ** 4
    B = su3.su3_field_bytes(ds)
    # weak scaling: the global lattice is (L, L, L, L*world), rank r owns the x3 slab r (section 8(e))
    gL = shard.weak_global_extents((L,) * 4, world)
    m0, m1 = shard.matrix_range(gL, 1, rank, world)
    assert m1 - m0 == nmat
    seed = su3gen.config_seed(5)

    # ---- seeded inputs, generated once on the host in fp64 (S10-S14) straight into pinned memory
    t0 = time.time()
    host = {}
    for name, fid in (("x", su3gen.FIELD_X), ("y", su3gen.FIELD_Y), ("w", su3gen.FIELD_W), ("v", su3gen.FIELD_V)):
        h = torch.empty(nmat * 9, dtype=torch.complex128, pin_memory=True)
        a = h.numpy().reshape(nmat, 3, 3)
        (su3gen.gaussian_field if name == "v" else su3gen.su3_field)(seed, fid, nmat, m0=m0, out=a)
        host[name] = h
    hz = [torch.empty(B, dtype=torch.uint8, pin_memory=True) for _ in range(3)]
    log("[rank %d] generated 4 x %d^4 fields (%.2f GB each) in %.1f s" % (rank, L, B / 1e9, time.time() - t0))

    def hbytes(t):
        return torch.view_as_real(t).view(-1).view(torch.uint8) if t.dtype == torch.complex128 else t

    f = {}
    for n_ in ("xs", "ys", "ws", "vs", "zs", "z4", "zb", "zc"):
        f[n_] = su3.alloc_field(ds, device=dev)
    for n_ in ("xv", "yv", "wv", "zv", "z3"):
        f[n_] = su3.alloc_field(dv, device=dev)
    for n_ in ("x", "y", "w", "v"):
        f[n_ + "s"].tensor.copy_(hbytes(host[n_]), non_blocking=True)
    torch.cuda.synchronize()

    rows = [  # (row, op, launch, field streams)
        ("A5 convert xs->xv", "convert", lambda: su3.su3_convert(f["xv"], f["xs"])),
        ("A5 convert ys->yv", "convert", lambda: su3.su3_convert(f["yv"], f["ys"])),
        ("A5 convert ws->wv", "convert", lambda: su3.su3_convert(f["wv"], f["ws"])),
        ("A1 mul scalar", "mul", lambda: su3.su3_mul(f["zs"], f["xs"], f["ys"])),
        ("A2 mul vector W=%d" % W64, "mul", lambda: su3.su3_mul(f["zv"], f["xv"], f["yv"])),
        ("A3 mul3 vector W=%d" % W64, "mul3", lambda: su3.su3_mul3(f["z3"], f["xv"], f["yv"], f["wv"])),
        ("A4 mul_add scalar", "mul_add", lambda: su3.su3_mul_add(f["z4"], f["xs"], f["ys"], f["vs"])),
        ("A5 convert zv->zb", "convert", lambda: su3.su3_convert(f["zb"], f["zv"])),
        ("A6 copy zs->zc", "copy", lambda: su3.su3_copy(f["zc"], f["zs"])),
    ]
    step_bytes = sum(STREAMS[op] for _, op, _ in rows) * B
    step_flops = sum(FLOPS[op] for _, op, _ in rows) * nmat

    def step(events=None):
        for i, (_, _, launch) in enumerate(rows):
            if events is not None:
                events[i].record()
            launch()
        if events is not None:
            events[len(rows)].record()

    # ---- device-resident timing: W warm-up steps, then exactly K steps, per-launch events inside
    clocks = ClockSampler(dev.index)   # sampled from here on: warm-up and timed steps are both under load
    t_warm = time.perf_counter()
    nwarm = 0
    while nwarm < max(args.warmup, 3) or time.perf_counter() - t_warm < 0.6:
        step()
        torch.cuda.synchronize()
        nwarm += 1
    barrier()
    K = args.steps
    evs = [[torch.cuda.Event(enable_timing=True) for _ in range(len(rows) + 1)] for _ in range(K)]
    n0 = su3.su3_launch_count()
    barrier()
    t_wall = time.perf_counter()
    for k in range(K):
        step(evs[k])
    torch.cuda.synchronize()
    if dist is not None:
        dist.barrier()
    t_wall = time.perf_counter() - t_wall
    launches = su3.su3_launch_count() - n0
    clk = clocks.stop()
    total_ms = evs[0][0].elapsed_time(evs[K - 1][len(rows)])
    row_ms = [float(np.mean([evs[k][i].elapsed_time(evs[k][i + 1]) for k in range(K)])) for i in range(len(rows))]
    # whole-job value: bytes of all ranks / max-over-ranks device time (independent shards, no collective)
    rate, total_ms, _ = shard.job_throughput(K * step_bytes, total_ms, dist, coll_dev)
    ms_per_step = total_ms / K
    value = rate / 1e9

    # ---- correctness tripwires on the full-size outputs (the parity tests proper are tests/ -m gpu)
    torch.cuda.synchronize()
    checks = {
        "vector_result_equals_scalar_result_bitwise": bool(torch.equal(f["zb"].tensor, f["zs"].tensor)),
        "copy_bitwise": bool(torch.equal(f["zc"].tensor, f["zs"].tensor)),
    }
    return dict(torch=torch, su3=su3, dist=dist, dev=coll_dev, f=f, host=host, hz=hz, rows=rows, row_ms=row_ms, B=B,
                nmat=nmat, step_bytes=step_bytes, step_flops=step_flops, ms_per_step=ms_per_step, value=value,
                launches=launches, clk=clk, checks=checks, nwarm=nwarm, info=info, t_wall=t_wall, barrier=barrier, step=step,
                hbytes=hbytes)


def time_calls(torch, fn, target_ms=2.0, batches=5, warm=3, graph_below_us=0.0):
    """SURVEY 8(d) protocol: warm-up calls, then `batches` batches of Nloop back-to-back calls between two
    CUDA events on the current stream; returns (min, median) ms per call and how the calls were issued.
    Calls shorter than `graph_below_us` are launch-bound from Python: their Nloop calls are captured once
    into a CUDA graph and the graph is replayed (the library's calls are capturable: no sync, no allocation)."""
    for _ in range(warm):
        fn()
    a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    a.record(); fn(); fn(); b.record(); b.synchronize()
    est = max(a.elapsed_time(b) / 2, 1e-3)
    nloop = int(min(1000, max(10, target_ms / est)))
    how = "stream"
    run = None
    if est * 1e3 < graph_below_us:
        g = torch.cuda.CUDAGraph()
        with torch.cuda.graph(g):
            for _ in range(nloop):
                fn()
        run, how = g.replay, "cuda_graph(%d calls)" % nloop
        run()
    per = []
    for _ in range(batches):
        a.record()
        if run is not None:
            run()
        else:
            for _ in range(nloop):
                fn()
        b.record(); b.synchronize()
        per.append(a.elapsed_time(b) / nloop)
    return float(min(per)), float(np.median(per)), how


def run_e2e(args, r, world):
    """The same step with HOST buffers: x, y in and the A1 result out through su3_mul_host (chunked, copy/compute
    overlapped inside the library); w, v in and the A2 (converted back), A3, A4 results out as plain async
    copies on the same stream.  Everything between the two events is inside the timed region."""
    torch, su3, f, host, hz, hbytes = r["torch"], r["su3"], r["f"], r["host"], r["hz"], r["hbytes"]
    B = r["B"]
    hx, hy, hw, hv = (hbytes(host[k]) for k in ("x", "y", "w", "v"))

    h2d_s, d2h_s = torch.cuda.Stream(), torch.cuda.Stream()

    def e2e_step():
        main = torch.cuda.current_stream()
        start = torch.cuda.Event(); start.record(main)
        # A1: x, y in and z out, chunked and overlapped inside the library; x, y stay resident for A2-A4
        su3.su3_mul_host(hz[0], hx, hy, f["zs"], f["xs"], f["ys"], chunks=E2E_CHUNKS)
        # w, v follow x, y on the H2D engine while the A1 result is already flowing back
        h2d_s.wait_event(start)
        with torch.cuda.stream(h2d_s):
            f["ws"].tensor.copy_(hw, non_blocking=True)
            ev_w = torch.cuda.Event(); ev_w.record(h2d_s)

        def result_to_host(field):
            ev = torch.cuda.Event(); ev.record(main)
            d2h_s.wait_event(ev)
            with torch.cuda.stream(d2h_s):
                hz[1].copy_(field.tensor, non_blocking=True)

        su3.su3_convert(f["xv"], f["xs"]); su3.su3_convert(f["yv"], f["ys"])
        su3.su3_mul(f["zv"], f["xv"], f["yv"])                                        # A2
        su3.su3_convert(f["zb"], f["zv"])
        result_to_host(f["zb"])
        su3.su3_copy(f["zc"], f["zs"])                                                # A6
        main.wait_event(ev_w)
        su3.su3_convert(f["wv"], f["ws"])
        su3.su3_mul3(f["z3"], f["xv"], f["yv"], f["wv"])                              # A3
        result_to_host(f["z3"])
        # A4 chunked through the library: v arrives chunk by chunk behind w, every chunk of x*y + v leaves at once
        su3.su3_eval_host(su3.SU3_OP_MUL_ADD, hz[2], None, None, hv, f["z4"], f["xs"], f["ys"], f["vs"], chunks=E2E_CHUNKS)
        done = torch.cuda.Event(); done.record(d2h_s)
        main.wait_event(done)

    n = max(2, min(args.steps, 5))
    e2e_step()
    r["barrier"]()
    a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    a.record()
    for _ in range(n):
        e2e_step()
    b.record()
    b.synchronize()
    from paper_1710_09409_b200 import shard
    rate, ms, _ = shard.job_throughput(r["step_bytes"], a.elapsed_time(b) / n, r["dist"], r["dev"])
    ok = bool(torch.equal(hz[0], f["zs"].tensor.cpu())) and bool(torch.equal(hz[2], f["z4"].tensor.cpu()))
    return {"value": rate / 1e9, "unit": UNIT, "h2d_bytes_per_step": 4 * B,
            "d2h_bytes_per_step": 4 * B, "ms_per_step": ms, "steps": n,
            "api": "su3_mul_host (A1), su3_eval_host (A4, x and y resident) + pinned async copies on side streams around su3_convert/su3_mul/su3_mul3/su3_copy",
            "host_result_matches_device": ok}


def run_ceilings_and_sweep(args, r):
    """Same-run ceilings (A6: own copy kernel, cudaMemcpyAsync D2D, the 2-read-1-write add) at the workload
    size, then the volume sweep of BASELINE.json configs[4]: z = x*y for L = 8..64, fp64/fp32, scalar/vector,
    warm protocol (Listing 3: same operands every call).  Operands are prefixes of the resident fields."""
    torch, su3, f, B = r["torch"], r["su3"], r["f"], r["B"]
    l2 = r["info"]["l2_bytes"]
    out = {}
    mn, md, _ = time_calls(torch, lambda: su3.su3_copy(f["zc"], f["zs"]))
    out["su3_copy"] = 2 * B / (mn * 1e-3) / 1e9
    mn, md, _ = time_calls(torch, lambda: f["zc"].tensor.copy_(f["zs"].tensor))
    out["memcpy_d2d"] = 2 * B / (mn * 1e-3) / 1e9
    mn, md, _ = time_calls(torch, lambda: su3.su3_add(f["zc"], f["xs"], f["ys"]))
    out["su3_add_2r1w"] = 3 * B / (mn * 1e-3) / 1e9
    ceiling = max(out["su3_copy"], out["memcpy_d2d"])
    out["bar_denominator"] = ceiling
    if args.no_sweep:
        return out, []
    # fp32 copies of x, y in both layouts (input preparation only: rounding fp64 -> fp32, S16)
    x32 = f["xs"].tensor.view(torch.float64).to(torch.float32)
    y32 = f["ys"].tensor.view(torch.float64).to(torch.float32)
    d32s = su3.make_desc(args.L, prec=su3.SU3_F32)
    d32v = su3.make_desc(args.L, prec=su3.SU3_F32, layout=su3.SU3_VECTOR, W=W32)
    fx32s, fy32s = su3.su3_field_wrap(d32s, x32.view(torch.uint8)), su3.su3_field_wrap(d32s, y32.view(torch.uint8))
    fx32v, fy32v = su3.alloc_field(d32v), su3.alloc_field(d32v)
    su3.su3_convert(fx32v, fx32s); su3.su3_convert(fy32v, fy32s)
    src = {(8, 0): (f["xs"], f["ys"], f["zc"]), (8, 1): (f["xv"], f["yv"], f["zc"]),
           (4, 0): (fx32s, fy32s, f["zc"]), (4, 1): (fx32v, fy32v, f["zc"])}
    # f1 (Fig. 4): vector-length sweep at a fixed HBM-bound volume, fp32 complex.
    # The paper's GPUs plateaued only at W = 16 because block = one vector; here bandwidth is flat in W.
    wsweep = []
    Lw = min(args.L, 48)
    for Wv in (1, 2, 4, 8, 16, 32):
        dsw = su3.make_desc(Lw, prec=su3.SU3_F32)
        dw = su3.make_desc(Lw, prec=su3.SU3_F32, layout=su3.SU3_VECTOR, W=Wv)
        nbw = su3.su3_field_bytes(dw)
        xs_w = su3.su3_field_wrap(dsw, x32[:nbw // 4].view(torch.uint8))
        ys_w = su3.su3_field_wrap(dsw, y32[:nbw // 4].view(torch.uint8))
        xw, yw, zw = su3.alloc_field(dw), su3.alloc_field(dw), su3.alloc_field(dw)
        su3.su3_convert(xw, xs_w); su3.su3_convert(yw, ys_w)
        mn, md, _ = time_calls(torch, lambda: su3.su3_mul(zw, xw, yw))
        wsweep.append({"W": Wv, "L": Lw, "prec": "f32", "simd": list(su3.su3_desc_normalize(dw).simd),
                       "us_min": mn * 1e3, "GBps": 3 * nbw / (mn * 1e-3) / 1e9,
                       "GFLOPps": FLOPS["mul"] * Lw ** 4 / (mn * 1e-3) / 1e9,
                       "frac_of_copy": 3 * nbw / (mn * 1e-3) / 1e9 / ceiling})
        del xw, yw, zw
    out["wsweep"] = wsweep
    sweep = []
    for Ls in (8, 12, 16, 24, 32, 48, 64):
        if Ls > args.L:
            continue
        for prec in (8, 4):
            for layout in (0, 1):
                W = 1 if layout == 0 else (W64 if prec == 8 else W32)
                d = su3.make_desc(Ls, prec=prec, layout=layout, W=W)
                nb = su3.su3_field_bytes(d)
                xs_, ys_, zs_ = src[(prec, layout)]
                fx = su3.su3_field_wrap(d, xs_.tensor[:nb]); fy = su3.su3_field_wrap(d, ys_.tensor[:nb])
                fz = su3.su3_field_wrap(d, zs_.tensor[:nb])
                mn, md, how = time_calls(torch, lambda: su3.su3_mul(fz, fx, fy), graph_below_us=60.0)
                gbs = 3 * nb / (mn * 1e-3) / 1e9
                regime = "L2-resident" if 3 * nb < 0.75 * l2 else ("HBM-bound" if 3 * nb > 2 * l2 else "straddles L2")
                cold = None
                if regime != "HBM-bound":
                    # "cold" protocol (S18): rotate through operand triples so that a call never finds its lines
                    # in L2; triple k = the k-th nb-sized slice of the resident 64^4-sized fields
                    nb_al = (nb + 255) // 256 * 256
                    ntrip = int(min(zs_.tensor.numel() // nb_al, xs_.tensor.numel() // nb_al, 2 * l2 // (3 * nb) + 2))
                    if ntrip * 3 * nb > 2 * l2:
                        trip = [tuple(su3.su3_field_wrap(d, t.tensor[k * nb_al:k * nb_al + nb]) for t in (zs_, xs_, ys_))
                                for k in range(ntrip)]
                        ctr = [0]

                        def rot():
                            z_, x_, y_ = trip[ctr[0] % ntrip]
                            ctr[0] += 1
                            su3.su3_mul(z_, x_, y_)
                        cmn, _, _ = time_calls(torch, rot, target_ms=4.0, warm=ntrip, graph_below_us=60.0)
                        cold = 3 * nb / (cmn * 1e-3) / 1e9
                sweep.append({"L": Ls, "prec": "f64" if prec == 8 else "f32", "layout": "scalar" if layout == 0 else "vector",
                              "W": W, "footprint_MB": 3 * nb / 1e6, "us_min": mn * 1e3, "us_median": md * 1e3, "issued": how,
                              "GBps": gbs, "GFLOPps": FLOPS["mul"] * Ls ** 4 / (mn * 1e-3) / 1e9, "regime": regime, "cold_GBps": cold,
                              "frac_of_copy": gbs / ceiling if regime == "HBM-bound" else None})
    return out, sweep


def run_next_rows(args, r):
    """SURVEY 8(f) rows beyond A1-A6, measured at an HBM-bound volume (48^4, fp64 scalar and vector W=4) with the
    same protocol: f2 the one-pass expression evaluator, f3 Cshift and the shifted product."""
    torch, su3, f = r["torch"], r["su3"], r["f"]
    Ln = min(args.L, 48)
    out = {"L": Ln, "prec": "f64", "expr": [], "shift": []}
    for layout, W, names in ((0, 1, ("xs", "ys", "ws", "vs")), (1, W64, ("xv", "yv", "wv", "z3"))):
        d = su3.make_desc(Ln, layout=layout, W=W)
        nb = su3.su3_field_bytes(d)
        ops = [su3.su3_field_wrap(d, f[n].tensor[:nb]) for n in names]
        z = su3.su3_field_wrap(d, f["zc"].tensor[:nb])
        lay = "scalar" if layout == 0 else "vector W=%d" % W
        for prog in ("01*", "01*2*", "01*2+", "01+01*+", "01*23*+", "01+2+3+"):
            n = max(int(c) for c in prog if c.isdigit()) + 1
            st, fl = su3.su3_expr_cost(prog, n)
            mn, _, _ = time_calls(torch, lambda: su3.su3_expr(z, prog, ops[:n]))
            out["expr"].append({"program": prog, "layout": lay, "streams": st, "flops_per_matrix": fl,
                                "GBps": st * nb / (mn * 1e-3) / 1e9, "GFLOPps": fl * Ln ** 4 / (mn * 1e-3) / 1e9})
        for dim in range(4):
            mn, _, _ = time_calls(torch, lambda: su3.su3_cshift(z, ops[1], dim, 1))
            mn2, _, _ = time_calls(torch, lambda: su3.su3_mul_shift(z, ops[0], ops[1], dim, 1))
            out["shift"].append({"dim": dim, "disp": 1, "layout": lay, "cshift_GBps": 2 * nb / (mn * 1e-3) / 1e9,
                                 "mul_shift_GBps": 3 * nb / (mn2 * 1e-3) / 1e9,
                                 "mul_shift_GFLOPps": FLOPS["mul"] * Ln ** 4 / (mn2 * 1e-3) / 1e9})
    # BASELINE.json configs[2] and configs[3] as bench points (their parity is in tests/test_gpu_fullsize.py)
    out["configs"] = []
    if args.L >= 48:
        d3s, d3v = su3.make_desc(32, n_lorentz=4), su3.make_desc(32, n_lorentz=4, layout=1, W=W64)
        nb3 = su3.su3_field_bytes(d3s)
        for d3, lay, (a_, b_) in ((d3s, "scalar", ("xs", "ys")), (d3v, "vector W=%d" % W64, ("xv", "yv"))):
            fa, fb, fz = (su3.su3_field_wrap(d3, f[n_].tensor[:nb3]) for n_ in (a_, b_, "zc"))
            mn, _, _ = time_calls(torch, lambda: su3.su3_mul(fz, fa, fb))
            out["configs"].append({"config": "cfg3: 32^4 x 4 Lorentz fp64, mul, " + lay, "GBps": 3 * nb3 / (mn * 1e-3) / 1e9,
                                   "GFLOPps": FLOPS["mul"] * 4 * 32 ** 4 / (mn * 1e-3) / 1e9})
        d4 = su3.make_desc(48, prec=su3.SU3_F32, layout=1, W=W32)
        nb4 = su3.su3_field_bytes(d4)
        f4 = [su3.su3_field_wrap(d4, f[n_].tensor[:nb4]) for n_ in ("xv", "yv", "wv", "zc")]   # fp64 bytes read as fp32:
        for fld in f4[:3]:                                                                      # make them finite numbers
            fld.tensor.view(torch.float32).normal_()
        for opn, fn in (("mul3", su3.su3_mul3), ("mul_add", su3.su3_mul_add)):
            mn, _, _ = time_calls(torch, lambda: fn(f4[3], f4[0], f4[1], f4[2]))
            out["configs"].append({"config": "cfg4: 48^4 fp32 vector W=%d, %s" % (W32, opn), "GBps": 4 * nb4 / (mn * 1e-3) / 1e9,
                                   "GFLOPps": FLOPS[opn] * 48 ** 4 / (mn * 1e-3) / 1e9})
    # the paper's Listing 2 on real scalar fields: v3 = v1+v2 and v3 = v1+v2+v1*v2 (3 streams of 8 / 4 B per element)
    out["listing2"] = []
    for prec in (8, 4):
        dr = su3.make_desc(Ln, n_lorentz=4, prec=prec)
        nr = su3.su3_real_bytes(dr)
        reps = max(1, (1 << 29) // nr)                       # batch enough copies of the field to stream >= 0.5 GB each
        dbig = su3.make_desc((Ln, Ln, Ln, Ln * reps), n_lorentz=4, prec=prec)
        nbig = su3.su3_real_bytes(dbig)
        v1, v2, v3 = (su3.su3_real_wrap(dbig, f[n_].tensor[:nbig]) for n_ in ("xs", "ys", "zc"))
        su3.su3_fill(v1, 1.0); su3.su3_fill(v2, 2.0)
        for prog, flops in (("01+", 1), ("01+01*+", 3)):
            mn, _, _ = time_calls(torch, lambda: su3.su3_expr(v3, prog, [v1, v2]))
            ok = bool((v3.tensor.view(torch.float64 if prec == 8 else torch.float32) == (3.0 if prog == "01+" else 5.0)).all())
            out["listing2"].append({"program": prog, "prec": "f64" if prec == 8 else "f32", "reals": nbig // prec,
                                    "GBps": 3 * nbig / (mn * 1e-3) / 1e9, "GFLOPps": flops * (nbig // prec) / (mn * 1e-3) / 1e9,
                                    "value_is_the_papers": ok})
    # f4: colour vectors, y = U.psi (66 flops, 240 B fp64 / 120 B fp32 per site)
    out["matvec"] = []
    for prec, layout, W in ((8, 0, 1), (8, 1, W64), (4, 0, 1), (4, 1, W32)):
        d = su3.make_desc(Ln, prec=prec, layout=layout, W=W)
        U = su3.su3_field_wrap(d, f["xs"].tensor[:su3.su3_field_bytes(d)])      # bandwidth is data-independent
        nv = su3.su3_vec_bytes(d)
        psi, yv = su3.su3_vec_wrap(d, f["ys"].tensor[:nv]), su3.su3_vec_wrap(d, f["zc"].tensor[:nv])
        mn, _, _ = time_calls(torch, lambda: su3.su3_matvec(yv, U, psi))
        nb = su3.su3_field_bytes(d) + 2 * nv
        out["matvec"].append({"prec": "f64" if prec == 8 else "f32", "layout": "scalar" if layout == 0 else "vector W=%d" % W,
                              "GBps": nb / (mn * 1e-3) / 1e9, "GFLOPps": 66 * Ln ** 4 / (mn * 1e-3) / 1e9})
    return out


def profile_pass(args):
    """One launch of every kernel variant at an HBM-bound size (inputs: Gaussian reals -- bandwidth and the
    counters ncu reads do not depend on the values).  Prints one JSON line with the launch count."""
    import torch

    import paper_1710_09409_b200 as su3
    torch.cuda.set_device(0)
    L = min(args.L, 48)
    n0 = su3.su3_launch_count()
    order = []
    for prec, W in ((su3.SU3_F64, W64), (su3.SU3_F32, W32)):
        dt = torch.float64 if prec == su3.SU3_F64 else torch.float32
        ds, dv = su3.make_desc(L, prec=prec), su3.make_desc(L, prec=prec, layout=su3.SU3_VECTOR, W=W)
        xs, ys, ws, zs = (su3.alloc_field(ds) for _ in range(4))
        xv, yv, wv, zv = (su3.alloc_field(dv) for _ in range(4))
        for fld in (xs, ys, ws):
            fld.tensor.view(dt).normal_()
        for dst, src in ((xv, xs), (yv, ys), (wv, ws)):
            su3.su3_convert(dst, src)
        order.append("convert s->v x3")
        for name, (x, y, w, z) in (("scalar", (xs, ys, ws, zs)), ("vector", (xv, yv, wv, zv))):
            for path, pname in ((1, "pipe"), (2, "direct"), (3, "warp")):
                su3.su3_tune_set(path=path)
                su3.su3_mul(z, x, y); su3.su3_mul3(z, x, y, w); su3.su3_mul_add(z, x, y, w)
                order.append("%s %s: mul mul3 mul_add" % (name, pname))
            su3.su3_tune_set(path=1)
            su3.su3_add(z, x, y); su3.su3_copy(z, x)
            su3.su3_tune_set(path=2)
            su3.su3_add(z, x, y); su3.su3_copy(z, x)
            su3.su3_tune_set()
            su3.su3_expr(z, "01+01*+", [x, y]); su3.su3_expr(z, "01*23*+", [x, y, w, x])
            su3.su3_cshift(z, y, 0, 1); su3.su3_cshift(z, y, 3, 1); su3.su3_mul_shift(z, x, y, 1, 1)
            psi = su3.su3_vec_wrap(x.desc, w.tensor[:su3.su3_vec_bytes(x.desc)])
            yv_ = su3.su3_vec_wrap(x.desc, z.tensor[:su3.su3_vec_bytes(x.desc)])
            su3.su3_matvec(yv_, x, psi)
        su3.su3_convert(zs, zv)
        torch.cuda.synchronize()
        del xs, ys, ws, zs, xv, yv, wv, zv
        torch.cuda.empty_cache()
    print(json.dumps({"profile_pass": True, "L": L, "launches": su3.su3_launch_count() - n0}), flush=True)


def main():
    args = parse_args()
    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))
    # torchrun exports OMP_NUM_THREADS=1; the host-side generator and the oracle (gcc/OpenMP libraries loaded later)
    # should still use the box's cores: all of them for the reference arm (rank 0 alone works), a fair share otherwise
    if world > 1 and os.environ.get("OMP_NUM_THREADS") == "1":
        ncpu = os.cpu_count() or 1
        os.environ["OMP_NUM_THREADS"] = str(ncpu if args.impl == "reference" else max(1, ncpu // world))
    if args.impl == "reference":
        run_reference(args, rank)
        return
    if args.profile_pass:
        if rank == 0:
            profile_pass(args)
        return
    if world != args.gpus:
        log("note: --gpus %d but WORLD_SIZE=%d; using WORLD_SIZE (launch N>1 with torch.distributed.run)" % (args.gpus, world))
    r = run_ours(args, rank, world, local_rank)
    torch = r["torch"]
    e2e = None if args.no_e2e else run_e2e(args, r, world)
    ceilings, sweep = ({}, [])
    next_rows = None
    if rank == 0:
        ceilings, sweep = run_ceilings_and_sweep(args, r)
        if not args.no_sweep:
            next_rows = run_next_rows(args, r)
    peak, peak_src = measured_peak()
    B, nmat = r["B"], r["nmat"]
    ops = []
    for (name, op, _), ms in zip(r["rows"], r["row_ms"]):
        gbs = STREAMS[op] * B / (ms * 1e-3) / 1e9
        ops.append({"row": name, "ms": ms, "GBps": gbs, "GFLOPps": FLOPS[op] * nmat / (ms * 1e-3) / 1e9,
                    "frac_of_measured_peak": gbs / peak,
                    "frac_of_copy": gbs / ceilings["bar_denominator"] if ceilings else None})
    a1 = ops[3]
    # nominal pin-rate peak from device properties: memory clock x 2 (DDR) x bus width / 8
    pin_rate = r["info"]["mem_clock_khz"] * 1e3 * 2 * r["info"]["bus_width_bits"] / 8 / 1e9
    roofline = {"bound": "hbm", "kernel": "su3_pipe_kernel<double,W=1,OP_MUL> (row A1, z=x*y fp64 scalar)",
                "achieved": a1["GBps"], "peak": peak, "unit": "GB/s", "frac": a1["GBps"] / peak, "peak_source": peak_src,
                "algorithmic_bytes_per_launch": 3 * B, "avg_launch_ms": a1["ms"],
                "frac_of_same_run_copy": a1["frac_of_copy"], "pin_rate_peak": pin_rate, "frac_of_pin_rate_peak": a1["GBps"] / pin_rate,
                # dram__bytes_read.sum + dram__bytes_write.sum of this launch at 64^4, from the one ncu --set full
                # capture summarised in profiles/r01_pipe_kernel_full.md (4.831918 + 2.385510 GB)
                "traffic": 7217428000 if args.L == 64 else None,
                "traffic_source": "profiles/r01_pipe_kernel_full.md (ncu --set full, per launch)"}
    cpu = None
    if rank == 0 and not args.no_cpu:
        Lc = min(args.cpu_L, args.L)
        times, nbytes, threads = oracle_step(Lc, 3)
        cpu = {"value": nbytes / min(times) / 1e9, "unit": UNIT, "cores": threads, "kind": "oracle",
               "sample": "rows A1-A6 on a %d^4 fp64 lattice (a smaller point of the same sweep), best of 3 passes" % Lc}
        t1, nb1, _ = oracle_step(min(Lc, 24), 1, threads=1)
        cpu["one_thread_value"] = nb1 / min(t1) / 1e9
        cpu["one_thread_sample"] = "the same rows on a %d^4 lattice, 1 thread, 1 pass" % min(Lc, 24)
    if r["dist"] is not None:
        r["dist"].barrier()
        r["dist"].destroy_process_group()
    if rank != 0:
        return
    line = {
        "metric": METRIC, "value": r["value"], "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": args.warmup, "warmup_steps_run": r["nwarm"],
        "ms_per_step": r["ms_per_step"], "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
        "dtype": "f64", "data": "synthetic",
        "config": {"workload": "BASELINE.json configs[4] top point: %d^4 lattice per GPU (%d matrices, %.3f GB per field), "
                               "fp64 complex, scalar + vector(W=%d) layouts, rows A1-A6 per step" % (args.L, nmat, B / 1e9, W64),
                   "L": args.L, "step_bytes": r["step_bytes"], "step_flops": r["step_flops"],
                   "l2_policy": "inputs larger than L2 (every launch streams >= %.1f GB; L2 = %.0f MB)" % (2 * B / 1e9, r["info"]["l2_bytes"] / 1e6),
                   "parallelism": "independent x3 slabs, no collective" if world > 1 else "single GPU"},
        "GFLOPps": world * r["step_flops"] / (r["ms_per_step"] * 1e-3) / 1e9,
        "gpu_launches": r["launches"], "clocks": r["clk"], "e2e": e2e, "roofline": roofline, "cpu_baseline": cpu,
        "ops": ops, "ceilings_GBps": {k: v for k, v in ceilings.items() if k != "wsweep"},
        "wsweep": ceilings.get("wsweep"), "next_rows": next_rows, "sweep": sweep, "checks": r["checks"],
        "wall_s_timed_region": r["t_wall"],
        # the paper's own numbers for z = x*y, as context only (other hardware, fp32, volumes unstated)
        "paper_context": {"hardware": "NVIDIA GTX 1080, 288 GB/s peak, ~240 GB/s sustainable (P:156)",
                          "z=x*y scalar AoS layout, CUDA/Jitify, no coalesced_ptr": "~120 GB/s (about half of sustainable)",
                          "z=x*y with coalesced_ptr (AoS -> AoSoAoS)": "saturates the memory bandwidth (~240 GB/s)",
                          "vector layout on GP100/V100": "follows the STREAM triad; plateau only at 16 threads per block (P:199-203)"},
    }
    print(json.dumps(line), flush=True)


if __name__ == "__main__":
    main()
