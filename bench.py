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
    ap.add_argument("--halo", action="store_true",
                    help="N > 1 with one GPU per rank (NCCL) only, opt-in: also time the one exchange step of the path, Cshift "
                         "along x3 across the slabs (halo.SlabShift: face pack -> NCCL send/recv || local shift -> unpack), and "
                         "report it beside the local su3_cshift under \"halo\"")
    ap.add_argument("--profile-pass", action="store_true",
                    help="launch every kernel variant of the library once at 48^4 (no timing): the command ncu wraps "
                         "for profiles/*_all_kernels.md")
    ap.add_argument("--profile-knee", action="store_true",
                    help="three back-to-back z = x*y calls per configuration at the knee of the volume sweep (24^4 fp64, 28^4 and "
                         "32^4 fp32, scalar and vector; footprints 0.6-2 x L2), no timing: the command ncu wraps with "
                         "--cache-control none for profiles/*_knee.md (the third call of each triple sees the L2 state the "
                         "warm protocol of the sweep sees)")
    return ap.parse_args()


def measured_peak():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    try:
        with open(p) as f:
            return float(json.load(f)["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)"
    except Exception:
        return 6650.0, "fallback (B200_PROFILING.md: 6.65 TB/s)"


# ---------------------------------------------------------------------------- the oracle legs
class OracleStep:
    """One step (rows A1-A6; A6 is a memcpy) by the oracle, as it stands, on an L^4 fp64 lattice.  Inputs come from
    su3gen (or from the caller: flat fp64 arrays in logical order); every output buffer is allocated once and
    first-touched by an untimed pass, so the timed passes contain the oracle's loops and nothing else."""

    def __init__(self, L, inputs=None, threads=None):
        import oracle
        import su3gen
        self.oracle = oracle
        if threads:
            oracle.set_num_threads(threads)
        self.gs, self.gv = oracle.Geom(L), oracle.Geom(L, layout=oracle.su3_oracle.VECTOR, W=W64)
        n = self.gs.nmat
        self.n = n
        if inputs is None:
            seed = su3gen.config_seed(5)
            inputs = [su3gen.su3_field(seed, f, n).view(np.float64).reshape(-1) for f in (0, 1, 2)]
            inputs.append(su3gen.gaussian_field(seed, 3, n).view(np.float64).reshape(-1))
        self.xs, self.ys, self.ws, self.vs = inputs
        self.out = {k: np.empty(n * 18, dtype=np.float64) for k in ("xv", "yv", "wv", "zs", "zv", "z3", "z4", "zb", "zc")}
        self.bytes = 24 * n * 144          # S9's accounting: 24 field streams
        self.threads = oracle.num_threads()
        self.run()                         # first touch of the outputs with the loops' own OpenMP schedule

    def run(self):
        o, b, gs, gv = self.oracle, self.out, self.gs, self.gv
        t0 = time.perf_counter()
        o.convert(gv, gs, self.xs, out=b["xv"]); o.convert(gv, gs, self.ys, out=b["yv"]); o.convert(gv, gs, self.ws, out=b["wv"])
        o.mul(gs, self.xs, self.ys, out=b["zs"])
        o.mul(gv, b["xv"], b["yv"], out=b["zv"])
        o.mul3(gv, b["xv"], b["yv"], b["wv"], out=b["z3"])
        o.mul_add(gs, self.xs, self.ys, self.vs, out=b["z4"])
        o.convert(gs, gv, b["zv"], out=b["zb"])
        np.copyto(b["zc"], b["zs"])
        return time.perf_counter() - t0

    def check(self):
        assert np.array_equal(self.out["zb"], self.out["zs"]) and np.array_equal(self.out["zc"], self.out["zs"])


REF_BUDGET_S = 240.0   # --impl reference: the whole run (W + K passes) should end within a few minutes


def run_reference(args, rank):
    """--impl reference: the oracle on the host cores, same metric/config.  Every step is one pass of rows A1-A6 at the
    WORKLOAD's own L whenever (W + K) passes fit the time budget (64^4: a few seconds per pass); otherwise a smaller
    point of the same sweep serves as the bounded sample, and `same_config` says so."""
    if rank != 0:
        return
    L = args.L
    st = OracleStep(L)
    t1 = st.run()
    total = args.warmup + args.steps
    while L > 16 and total * t1 > REF_BUDGET_S:
        L = {64: 48, 48: 32, 32: 24, 24: 16}.get(L, 16)
        del st
        st = OracleStep(L)
        t1 = st.run()
    times = [st.run() for _ in range(total)]
    st.check()
    timed = times[args.warmup:]
    sec = sum(timed) / len(timed)
    val = st.bytes / sec / 1e9
    same = L == args.L
    sample = ("every step = one pass of rows A1-A6 on the workload's own %d^4 fp64 lattice" % L if same else
              "every step = rows A1-A6 on a %d^4 fp64 lattice (a smaller point of the same sweep; workload %d^4)" % (L, args.L))
    print(json.dumps({
        "impl": "reference", "metric": METRIC, "value": val, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": sec * 1e3, "higher_is_better": True, "scaling": "weak",
        "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {"workload": "BASELINE.json configs[4] top point: %d^4 lattice, fp64 complex, scalar + vector(W=%d) layouts, "
                               "rows A1-A6 per step" % (args.L, W64), "L": args.L, "sample_L": L, "same_config": same},
        "cpu_baseline": {"value": val, "unit": UNIT, "cores": st.threads, "kind": "oracle", "sample": sample},
        "e2e": {"value": val, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
    }), flush=True)


def run_cpu_baseline(args, host):
    """cpu_baseline leg (rank 0, N = 1): the oracle on the box's host cores.  `value` = one step (rows A1-A6) at the
    workload's own L, all cores, best of 2 after a first-touch pass; beside it `z = x*y` (and the fused expressions of
    config 4) per BASELINE.json config, best of 3, with the bytes the oracle really moves (fp32 configs: fp32 in, fp64
    out = 288 B per matrix for mul), the one-thread figure, and a host STREAM triad."""
    import oracle
    VEC = oracle.su3_oracle.VECTOR
    L = args.L
    flat = [host[k].numpy().view(np.float64).reshape(-1) for k in ("x", "y", "w", "v")]
    st = OracleStep(L, inputs=flat)
    t = min(st.run(), st.run())
    st.check()
    cpu = {"value": st.bytes / t / 1e9, "unit": UNIT, "cores": st.threads, "kind": "oracle",
           "sample": "one step = rows A1-A6 on the workload's own %d^4 fp64 lattice, all cores, best of 2 passes after a "
                     "first-touch pass" % L, "ms_per_step": t * 1e3}
    del st

    def best_of(fn, reps=3):
        fn()
        return min(_timeit(fn) for _ in range(reps))

    def _timeit(fn):
        t0 = time.perf_counter()
        fn()
        return time.perf_counter() - t0

    per = []

    def mul_point(name, Lc, nl, prec, layout, W, ops=("mul",)):
        g = oracle.Geom(Lc, nl=nl, layout=layout, W=W)
        gs = oracle.Geom(Lc, nl=nl)
        n = g.nmat
        if n * 18 > flat[0].size:
            return
        dt = np.float64 if prec == 8 else np.float32
        used = {0, 1} | ({2} if "mul3" in ops else set()) | ({3} if "mul_add" in ops else set())
        # a prefix of the resident fields: timing is data-independent
        ins = [np.ascontiguousarray(a[:n * 18], dtype=dt) if k in used else None for k, a in enumerate(flat)]
        if layout == VEC:
            ins = [oracle.convert(g, gs, a) if a is not None else None for a in ins]
        out = np.zeros(n * 18, dtype=np.float64)
        for op in ops:
            fn = {"mul": lambda: oracle.mul(g, ins[0], ins[1], out=out),
                  "mul3": lambda: oracle.mul3(g, ins[0], ins[1], ins[2], out=out),
                  "mul_add": lambda: oracle.mul_add(g, ins[0], ins[1], ins[3], out=out)}[op]
            sec = best_of(fn)
            nin = 2 if op == "mul" else 3
            moved = n * (nin * 18 * prec + 144)                  # inputs in storage precision, fp64 result
            per.append({"config": name, "op": op, "GBps": moved / sec / 1e9, "GFLOPps": FLOPS[op] * n / sec / 1e9,
                        "bytes_per_matrix": nin * 18 * prec + 144, "ms": sec * 1e3})

    mul_point("cfg1: 8^4 fp64 scalar", 8, 1, 8, 0, 1)
    mul_point("cfg2: 16^4 fp64 scalar", 16, 1, 8, 0, 1)
    mul_point("cfg2: 16^4 fp64 vector W=%d" % W64, 16, 1, 8, VEC, W64)
    mul_point("cfg3: 32^4 x 4 Lorentz fp64 scalar", 32, 4, 8, 0, 1)
    mul_point("cfg3: 32^4 x 4 Lorentz fp64 vector W=%d" % W64, 32, 4, 8, VEC, W64)
    mul_point("cfg4: 48^4 fp32 vector W=%d" % W32, 48, 1, 4, VEC, W32, ops=("mul3", "mul_add"))
    mul_point("cfg5: 48^4 fp64 scalar", 48, 1, 8, 0, 1)
    mul_point("cfg5: %d^4 fp64 scalar" % L, L, 1, 8, 0, 1)
    mul_point("cfg5: %d^4 fp32 vector W=%d" % (L, W32), L, 1, 4, VEC, W32)
    cpu["per_config"] = per
    cpu["stream_triad_GBps"] = oracle.stream_triad(1 << 27)
    nthreads = oracle.num_threads()
    oracle.set_num_threads(1)
    try:
        L1 = min(L, 32)
        g1 = oracle.Geom(L1)
        n1 = g1.nmat
        out1 = np.zeros(n1 * 18, dtype=np.float64)
        sec = best_of(lambda: oracle.mul(g1, flat[0][:n1 * 18], flat[1][:n1 * 18], out=out1))
        cpu["one_thread"] = {"op": "mul", "sample": "z = x*y on a %d^4 fp64 lattice, 1 thread, best of 3" % L1,
                             "GBps": 3 * n1 * 144 / sec / 1e9, "GFLOPps": FLOPS["mul"] * n1 / sec / 1e9,
                             "stream_triad_GBps": oracle.stream_triad(1 << 25)}
    finally:
        oracle.set_num_threads(nthreads)
    return cpu


# ---------------------------------------------------------------------------- clocks during the timed region
CLOCK_Q = ("index,clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.active,clocks_event_reasons.hw_slowdown,"
           "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
           "clocks_event_reasons.sw_power_cap,clocks.mem,clocks.max.mem,name")


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
        sm, smax, reasons, power, mem, memmax, name = [], [], set(), [], [], [], None
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for line in self.f:
            c = [t.strip() for t in line.split(",")]
            if len(c) < 9:
                continue
            try:
                sm.append(float(c[1])); smax.append(float(c[2])); power.append(float(c[3]))
            except ValueError:
                continue
            if len(c) >= 12:
                try:
                    mem.append(float(c[9])); memmax.append(float(c[10])); name = c[11]
                except ValueError:
                    pass
            for nm, v in zip(names, c[5:9]):
                if v.lower().startswith("active"):
                    reasons.add(nm)
        self.f.close()
        os.unlink(self.f.name)
        if not sm:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["no samples"]}
        return {"sm_mhz": float(np.median(sm)), "sm_max_mhz": max(smax), "power_w_max": max(power),
                "mem_mhz": float(np.median(mem)) if mem else None, "mem_max_mhz": max(memmax) if memmax else None,
                "gpu_name": name, "samples": len(sm), "reasons": sorted(reasons)}


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
    gpu_name, _ = su3.su3_device_name()
    return dict(torch=torch, su3=su3, dist=dist, dev=coll_dev, gpu_name=gpu_name, f=f, host=host, hz=hz, rows=rows, row_ms=row_ms, B=B,
                nmat=nmat, step_bytes=step_bytes, step_flops=step_flops, ms_per_step=ms_per_step, value=value,
                launches=launches, clk=clk, checks=checks, nwarm=nwarm, info=info, t_wall=t_wall, barrier=barrier, step=step,
                hbytes=hbytes)


def time_calls(torch, fn, target_ms=2.0, batches=10, warm=3, graph_below_us=0.0):
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


def run_halo(args, r, world, rank):
    """The exchange step of the multi-GPU path, timed on every rank with CUDA events, max over ranks.
    A tripwire checks the data that crossed: the last x3 plane of rank r's result must equal, bit for bit and in both
    layouts, the first plane of rank r+1's input."""
    torch, su3, f, dist = r["torch"], r["su3"], r["f"], r["dist"]
    from paper_1710_09409_b200 import halo, shard
    sh = halo.SlabShift(halo.DistComm(dist))
    out = []
    for name_y, name_z, lay in (("ys", "zc", "scalar"), ("yv", "zv", "vector W=%d" % W64)):
        y, z = f[name_y], f[name_z]
        res = {"layout": lay}
        for label, fn in (("sharded", lambda: sh.cshift(z, y, 3, 1)), ("local_periodic", lambda: su3.su3_cshift(z, y, 3, 1))):
            for _ in range(3):
                fn()
            a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            r["barrier"]()
            a.record()
            for _ in range(10):
                fn()
            b.record(); b.synchronize()
            _, ms, _ = shard.job_throughput(1.0, a.elapsed_time(b) / 10, dist, r["dev"])
            res[label + "_ms"] = ms
            res[label + "_GBps_per_rank"] = 2 * y.nbytes / (ms * 1e-3) / 1e9
        # tripwire on the data that crossed, in BOTH layouts and over the whole plane: the last x3 plane of my result must be,
        # bit for bit, the first x3 plane of the next rank's input.  Planes are compared in the packed plane order
        # (su3_face_pack), which is the same for every layout; the next rank's plane arrives over a ring send/recv.
        try:
            sh.cshift(z, y, 3, 1)
            nb = su3.su3_face_bytes(y, 3, 1)
            first_in, last_out, nxt_in = (torch.empty(nb, dtype=torch.uint8, device=y.tensor.device) for _ in range(3))
            su3.su3_face_pack(first_in, y, 3, 0, 1)
            su3.su3_face_pack(last_out, z, 3, y.desc.L[3] - 1, 1)
            torch.cuda.synchronize()
            works = dist.batch_isend_irecv([dist.P2POp(dist.isend, first_in, (rank - 1) % world),
                                            dist.P2POp(dist.irecv, nxt_in, (rank + 1) % world)])
            for w in works:
                w.wait()
            torch.cuda.synchronize()
            ok = torch.tensor([1 if torch.equal(nxt_in, last_out) else 0], device=y.tensor.device)
            dist.all_reduce(ok, op=dist.ReduceOp.MIN)
            res["face_plane_bit_equal"] = bool(int(ok.item()) == 1)
        except Exception as e:  # the opt-in leg must not take the bench line down with it
            res["face_plane_bit_equal"] = None
            res["face_check_error"] = "%s: %s" % (type(e).__name__, e)
        out.append(res)
    return out


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
    # and the host results against the ORACLE on sampled matrices (A1: z = x*y, A4: z = x*y + v)
    import oracle
    nmat = r["nmat"]
    pick = np.unique(np.concatenate([np.random.default_rng(5).integers(0, nmat, 4000), [0, 1, nmat - 2, nmat - 1]]))
    small = oracle.Geom((len(pick), 1, 1, 1))
    sx, sy, sv = (host[k].numpy().reshape(nmat, 9)[pick].view(np.float64).reshape(-1) for k in ("x", "y", "v"))
    errs = []
    for hzk, ref in ((hz[0], oracle.mul(small, sx, sy)), (hz[2], oracle.mul_add(small, sx, sy, sv))):
        got = hzk.numpy().view(np.float64).reshape(nmat, 18)[pick]
        ref = ref.reshape(-1, 18)
        errs.append(float((np.abs(got - ref).max(axis=1) / np.abs(ref).max(axis=1)).max()))
    return {"value": rate / 1e9, "host_result_vs_oracle_sampled": {"matrices": int(len(pick)), "max_rel_err_A1": errs[0],
                                                                      "max_rel_err_A4": errs[1], "ok": bool(max(errs) <= 1e-12)}, "unit": UNIT, "h2d_bytes_per_step": 4 * B,
            "d2h_bytes_per_step": 4 * B, "ms_per_step": ms, "steps": n,
            "api": "su3_mul_host (A1), su3_eval_host (A4, x and y resident) + pinned async copies on side streams around su3_convert/su3_mul/su3_mul3/su3_copy",
            "host_result_matches_device": ok}


class Ceilings:
    """Same-run streaming ceilings at ANY field size (the paper draws its STREAM line across the whole footprint
    axis, Fig. 3): the library's own TMA copy kernel, cudaMemcpyAsync D2D (torch copy_) and the
    2-read-1-write add, timed with the sweep's own protocol on prefixes of resident fields; cached per size."""

    def __init__(self, torch, su3, a, b, c, l2):
        self.torch, self.su3, self.a, self.b, self.c, self.l2 = torch, su3, a, b, c, l2
        self.cache = {}

    def at(self, L, prec, nl=1):
        key = (L, prec, nl)
        if key in self.cache:
            return self.cache[key]
        torch, su3 = self.torch, self.su3
        d = su3.make_desc(L, n_lorentz=nl, prec=prec)
        nb = su3.su3_field_bytes(d)
        fa, fb, fc = (su3.su3_field_wrap(d, t.tensor[:nb]) for t in (self.a, self.b, self.c))
        out = {"L": L, "prec": "f64" if prec == 8 else "f32", "field_MB": nb / 1e6}
        mn, _, how = time_calls(torch, lambda: su3.su3_copy(fc, fa), graph_below_us=60.0)
        out["su3_copy"] = 2 * nb / (mn * 1e-3) / 1e9
        mn, _, _ = time_calls(torch, lambda: fc.tensor.copy_(fa.tensor), graph_below_us=60.0)
        out["memcpy_d2d"] = 2 * nb / (mn * 1e-3) / 1e9
        mn, _, _ = time_calls(torch, lambda: su3.su3_add(fc, fa, fb), graph_below_us=60.0)
        out["su3_add_2r1w"] = 3 * nb / (mn * 1e-3) / 1e9
        out["best_copy"] = max(out["su3_copy"], out["memcpy_d2d"])
        out["issued"] = how
        if 3 * nb <= 2 * self.l2:
            # cold protocol (S18) for the copy as well: rotate through (dst, src) pairs that together exceed 2 x L2
            nb_al = (nb + 255) // 256 * 256
            npair = int(min(self.a.tensor.numel() // nb_al, 2 * self.l2 // (2 * nb) + 2))
            if npair * 2 * nb > 2 * self.l2:
                pairs = [(su3.su3_field_wrap(d, self.c.tensor[k * nb_al:k * nb_al + nb]),
                          su3.su3_field_wrap(d, self.a.tensor[k * nb_al:k * nb_al + nb])) for k in range(npair)]
                ctr = [0]

                def rot():
                    dst, src = pairs[ctr[0] % npair]
                    ctr[0] += 1
                    su3.su3_copy(dst, src)
                cmn, _, _ = time_calls(torch, rot, target_ms=4.0, warm=npair, graph_below_us=60.0)
                out["su3_copy_cold"] = 2 * nb / (cmn * 1e-3) / 1e9
        self.cache[key] = out
        return out

    def fresh(self, L, prec):
        """best of su3_copy / D2D re-timed NOW (not cached): the boxes run under a power cap and drift by several per cent
        over the minutes a full run takes, so a block of rows is judged against a ceiling measured right before it"""
        torch, su3 = self.torch, self.su3
        d = su3.make_desc(L, prec=prec)
        nb = su3.su3_field_bytes(d)
        fa, fc = (su3.su3_field_wrap(d, t.tensor[:nb]) for t in (self.a, self.c))
        t1, _, _ = time_calls(torch, lambda: su3.su3_copy(fc, fa), batches=5, graph_below_us=60.0)
        t2, _, _ = time_calls(torch, lambda: fc.tensor.copy_(fa.tensor), batches=5, graph_below_us=60.0)
        return 2 * nb / (min(t1, t2) * 1e-3) / 1e9


def run_ceilings_and_sweep(args, r):
    """Same-run ceilings (A6) at the workload size and at EVERY sweep size, then the volume sweep of BASELINE.json
    configs[4]: z = x*y for L = 8..64, fp64/fp32, scalar/vector, warm protocol (Listing 3: same operands every call)
    and, below 2 x L2, cold protocol (rotating operands).  Operands are prefixes of the resident fields."""
    torch, su3, f, B = r["torch"], r["su3"], r["f"], r["B"]
    l2 = r["info"]["l2_bytes"]
    ceil = Ceilings(torch, su3, f["zs"], f["xs"], f["zc"], l2)
    r["ceil"] = ceil
    top = ceil.at(args.L, 8)
    out = {"su3_copy": top["su3_copy"], "memcpy_d2d": top["memcpy_d2d"], "su3_add_2r1w": top["su3_add_2r1w"],
           "bar_denominator": top["best_copy"]}
    ceiling = top["best_copy"]
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
    # A5 in fp32 rides along: the scalar <-> vector permutation is timed for every W, both directions.
    wsweep, conv32 = [], []
    for Lw in sorted({min(args.L, 48), args.L}):
        cw = ceil.at(Lw, 4)
        for Wv in (1, 2, 4, 8, 16, 32):
            dsw = su3.make_desc(Lw, prec=su3.SU3_F32)
            dw = su3.make_desc(Lw, prec=su3.SU3_F32, layout=su3.SU3_VECTOR, W=Wv)
            nbw = su3.su3_field_bytes(dw)
            xs_w = su3.su3_field_wrap(dsw, x32[:nbw // 4].view(torch.uint8))
            ys_w = su3.su3_field_wrap(dsw, y32[:nbw // 4].view(torch.uint8))
            xw, yw, zw = su3.alloc_field(dw), su3.alloc_field(dw), su3.alloc_field(dw)
            back = su3.su3_field_wrap(dsw, f["zc"].tensor[:nbw])
            su3.su3_convert(xw, xs_w); su3.su3_convert(yw, ys_w)
            if Wv >= 2:
                t_sv, _, _ = time_calls(torch, lambda: su3.su3_convert(xw, xs_w))
                t_vs, _, _ = time_calls(torch, lambda: su3.su3_convert(back, xw))
                ok = bool(torch.equal(back.tensor, xs_w.tensor))
                conv32.append({"L": Lw, "W": Wv, "prec": "f32", "scalar_to_vector_GBps": 2 * nbw / (t_sv * 1e-3) / 1e9,
                               "vector_to_scalar_GBps": 2 * nbw / (t_vs * 1e-3) / 1e9,
                               "frac_of_copy": [2 * nbw / (t * 1e-3) / 1e9 / cw["best_copy"] for t in (t_sv, t_vs)],
                               "round_trip_bit_exact": ok})
            if Lw == min(args.L, 48):
                mn, md, _ = time_calls(torch, lambda: su3.su3_mul(zw, xw, yw))
                wsweep.append({"W": Wv, "L": Lw, "prec": "f32", "simd": list(su3.su3_desc_normalize(dw).simd),
                               "us_min": mn * 1e3, "GBps": 3 * nbw / (mn * 1e-3) / 1e9,
                               "GFLOPps": FLOPS["mul"] * Lw ** 4 / (mn * 1e-3) / 1e9,
                               "frac_of_copy": 3 * nbw / (mn * 1e-3) / 1e9 / cw["best_copy"]})
            del xw, yw, zw
    out["wsweep"] = wsweep
    out["convert_f32"] = conv32
    sweep, by_size = [], []
    for Ls in (8, 12, 16, 24, 32, 48, 64):
        if Ls > args.L:
            continue
        for prec in (8, 4):
            c = ceil.at(Ls, prec)
            by_size.append(c)
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
                pl = su3.su3_launch_plan(d, 0)                      # the library's automatic choice at this point
                plan = pl["family"] if pl["family"] != "pipe" else "pipe tile %d depth %d l2 %s" % (
                    pl["tile"], pl["depth"], "pin %.1f MB/operand" % (pl["pin_bytes"] / 1e6) if pl["l2"] == "pin" else pl["l2"])
                sweep.append({"L": Ls, "prec": "f64" if prec == 8 else "f32", "layout": "scalar" if layout == 0 else "vector",
                              "W": W, "plan": plan, "footprint_MB": 3 * nb / 1e6, "us_min": mn * 1e3, "us_median": md * 1e3, "issued": how,
                              "GBps": gbs, "GFLOPps": FLOPS["mul"] * Ls ** 4 / (mn * 1e-3) / 1e9, "regime": regime, "cold_GBps": cold,
                              # against the SAME-SIZE ceilings of this run (warm: best of su3_copy / D2D; and the 2r1w add)
                              "frac_of_copy": gbs / c["best_copy"], "frac_of_add_2r1w": gbs / c["su3_add_2r1w"],
                              "cold_frac_of_copy": cold / c["su3_copy_cold"] if cold and c.get("su3_copy_cold") else None})
    out["by_size"] = by_size
    # The denominator of the latency-bound ramp (Fig. 3's left end): the library's smallest launch -- z = x*y on
    # a 2^4 lattice, 16 matrices, one block -- issued from the stream and replayed from a CUDA graph.  What an 8^4-16^4
    # call costs beyond this is the kernel's own time; the floor itself is launch latency, not the library's.
    d0 = su3.make_desc(2)
    nb0 = su3.su3_field_bytes(d0)
    f0 = [su3.su3_field_wrap(d0, t.tensor[:nb0]) for t in (f["zc"], f["xs"], f["ys"])]
    fl_stream, _, _ = time_calls(torch, lambda: su3.su3_mul(*f0))
    fl_graph, _, how = time_calls(torch, lambda: su3.su3_mul(*f0), graph_below_us=1e9)
    out["launch_floor_us"] = {"what": "su3_mul on a 2^4 lattice (16 matrices): the cost of one launch of this library",
                              "stream": fl_stream * 1e3, "graph_replay": fl_graph * 1e3, "graph": how}
    return out, sweep


def run_next_rows(args, r):
    """SURVEY 8(f) rows beyond A1-A6, measured at an HBM-bound volume (48^4, fp64 scalar and vector W=4) with the
    same protocol: f2 the one-pass expression evaluator, f3 Cshift and the shifted product."""
    torch, su3, f = r["torch"], r["su3"], r["f"]
    Ln = min(args.L, 48)
    c64, c32 = r["ceil"].at(Ln, 8)["best_copy"], r["ceil"].at(Ln, 4)["best_copy"]
    out = {"L": Ln, "prec": "f64", "copy_ceiling_GBps": {"f64": c64, "f32": c32}, "expr": [], "shift": [],
           "ceiling_protocol": "every block of rows (expr / shift per layout, listing2, matvec per precision) is divided by a copy "
                               "ceiling re-timed right before it (copy_now_GBps); copy_ceiling_GBps is the one timed with the sweep"}
    for layout, W, names in ((0, 1, ("xs", "ys", "ws", "vs")), (1, W64, ("xv", "yv", "wv", "z3"))):
        d = su3.make_desc(Ln, layout=layout, W=W)
        nb = su3.su3_field_bytes(d)
        ops = [su3.su3_field_wrap(d, f[n].tensor[:nb]) for n in names]
        z = su3.su3_field_wrap(d, f["zc"].tensor[:nb])
        lay = "scalar" if layout == 0 else "vector W=%d" % W
        c64 = r["ceil"].fresh(Ln, 8)
        # programs on the ahead-of-time menu (they run on the pipeline kernel), programs that are not (the interpreter),
        # and two menu programs forced through the interpreter (launch knob path = 3) for comparison
        for prog, force in (("01*", 0), ("01*2*", 0), ("01*2+", 0), ("01+01*+", 0), ("01*23*+", 0), ("01+2+3+", 0),
                            ("01*2*3*", 0), ("01*23**", 0), ("012**", 0), ("01*2*0*", 0), ("01*23*+0-", 0),
                            ("01+01*+", 1), ("01*23*+", 1), ("01*23**", 1)):
            n = max(int(c) for c in prog if c.isdigit()) + 1
            st, fl = su3.su3_expr_cost(prog, n)
            plan = su3.su3_expr_plan(prog, n)
            if force:
                su3.su3_tune_set(path=3)
            mn, _, _ = time_calls(torch, lambda: su3.su3_expr(z, prog, ops[:n]))
            su3.su3_tune_set()
            out["expr"].append({"program": prog, "layout": lay, "streams": st, "flops_per_matrix": fl,
                                "kernel": "interpreter" if force or plan == "interpreter" else "menu row %d" % plan[1],
                                "GBps": st * nb / (mn * 1e-3) / 1e9, "GFLOPps": fl * Ln ** 4 / (mn * 1e-3) / 1e9,
                                "copy_now_GBps": c64, "frac_of_copy": st * nb / (mn * 1e-3) / 1e9 / c64})
        c64 = r["ceil"].fresh(Ln, 8)
        for dim in range(4):
            mn, _, _ = time_calls(torch, lambda: su3.su3_cshift(z, ops[1], dim, 1))
            mn2, _, _ = time_calls(torch, lambda: su3.su3_mul_shift(z, ops[0], ops[1], dim, 1))
            out["shift"].append({"dim": dim, "disp": 1, "layout": lay, "cshift_GBps": 2 * nb / (mn * 1e-3) / 1e9,
                                 "mul_shift_GBps": 3 * nb / (mn2 * 1e-3) / 1e9, "copy_now_GBps": c64,
                                 "cshift_frac_of_copy": 2 * nb / (mn * 1e-3) / 1e9 / c64,
                                 "mul_shift_frac_of_copy": 3 * nb / (mn2 * 1e-3) / 1e9 / c64,
                                 "mul_shift_GFLOPps": FLOPS["mul"] * Ln ** 4 / (mn2 * 1e-3) / 1e9})
    # (e) the kernels of the multi-GPU shift: pack + unpack of the x3 face of 1 and 4 planes (bytes = 2 x face, each way)
    out["face"] = []
    for layout, W, name in ((0, 1, "xs"), (1, W64, "xv")):
        d = su3.make_desc(Ln, layout=layout, W=W)
        nb = su3.su3_field_bytes(d)
        x = su3.su3_field_wrap(d, f[name].tensor[:nb])
        z = su3.su3_field_wrap(d, f["zc"].tensor[:nb])
        for n in (1, 4):
            fb = su3.su3_face_bytes(x, 3, n)
            buf = torch.empty(fb, dtype=torch.uint8, device=x.tensor.device)
            t1, _, _ = time_calls(torch, lambda: su3.su3_face_pack(buf, x, 3, 0, n), graph_below_us=60.0)
            t2, _, _ = time_calls(torch, lambda: su3.su3_face_unpack(z, buf, 3, Ln - n, n), graph_below_us=60.0)
            out["face"].append({"layout": "scalar" if layout == 0 else "vector W=%d" % W, "planes": n, "face_MB": fb / 1e6,
                                "pack_us": t1 * 1e3, "unpack_us": t2 * 1e3, "pack_GBps": 2 * fb / (t1 * 1e-3) / 1e9,
                                "unpack_GBps": 2 * fb / (t2 * 1e-3) / 1e9})
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
        c64 = c32 = r["ceil"].fresh(Ln, prec)
        dr = su3.make_desc(Ln, n_lorentz=4, prec=prec)
        nr = su3.su3_real_bytes(dr)
        reps = max(1, min((1 << 29) // nr, f["zc"].nbytes // nr))   # batch copies of the field to stream up to 0.5 GB each (within the resident fields)
        dbig = su3.make_desc((Ln, Ln, Ln, Ln * reps), n_lorentz=4, prec=prec)
        nbig = su3.su3_real_bytes(dbig)
        v1, v2, v3 = (su3.su3_real_wrap(dbig, f[n_].tensor[:nbig]) for n_ in ("xs", "ys", "zc"))
        su3.su3_fill(v1, 1.0); su3.su3_fill(v2, 2.0)
        for prog, flops in (("01+", 1), ("01+01*+", 3)):
            mn, _, _ = time_calls(torch, lambda: su3.su3_expr(v3, prog, [v1, v2]))
            ok = bool((v3.tensor.view(torch.float64 if prec == 8 else torch.float32) == (3.0 if prog == "01+" else 5.0)).all())
            out["listing2"].append({"program": prog, "prec": "f64" if prec == 8 else "f32", "reals": nbig // prec,
                                    "GBps": 3 * nbig / (mn * 1e-3) / 1e9, "GFLOPps": flops * (nbig // prec) / (mn * 1e-3) / 1e9,
                                    "frac_of_copy": 3 * nbig / (mn * 1e-3) / 1e9 / (c64 if prec == 8 else c32),
                                    "value_is_the_papers": ok})
    # f4: colour vectors, y = U.psi (66 flops, 240 B fp64 / 120 B fp32 per site)
    out["matvec"] = []
    for prec, layout, W in ((8, 0, 1), (8, 1, W64), (4, 0, 1), (4, 1, W32)):
        if layout == 0:
            c64 = c32 = r["ceil"].fresh(Ln, prec)
        d = su3.make_desc(Ln, prec=prec, layout=layout, W=W)
        U = su3.su3_field_wrap(d, f["xs"].tensor[:su3.su3_field_bytes(d)])      # bandwidth is data-independent
        nv = su3.su3_vec_bytes(d)
        psi, yv = su3.su3_vec_wrap(d, f["ys"].tensor[:nv]), su3.su3_vec_wrap(d, f["zc"].tensor[:nv])
        mn, _, _ = time_calls(torch, lambda: su3.su3_matvec(yv, U, psi))
        nb = su3.su3_field_bytes(d) + 2 * nv
        out["matvec"].append({"prec": "f64" if prec == 8 else "f32", "layout": "scalar" if layout == 0 else "vector W=%d" % W,
                              "GBps": nb / (mn * 1e-3) / 1e9, "GFLOPps": 66 * Ln ** 4 / (mn * 1e-3) / 1e9,
                              "frac_of_copy": nb / (mn * 1e-3) / 1e9 / (c64 if prec == 8 else c32)})
    return out


def ncu_traffic(L, row="A1"):
    """dram__bytes_read.sum + dram__bytes_write.sum per launch of one kernel of the step (row A1, the dominant family, or
    A5, the largest single kernel): NOT measured in this run (no number is ever taken under a profiler here) but read
    from the committed ncu --set full summaries, whose headers name the command, the lattice and the commit they were
    captured at.  A line `traffic_bytes_per_launch = N (L = ..)` is row A1's, `traffic_bytes_per_launch[A5] = N (..)` row
    A5's; the newest round's file wins.  None if there is no capture for this L."""
    import glob
    import re
    tag = r"" if row == "A1" else r"\[%s\]" % re.escape(row)
    for path in sorted(glob.glob(os.path.join(ROOT, "profiles", "r*_full.md")), reverse=True):
        text = open(path).read()
        for m in re.finditer(r"traffic_bytes_per_launch" + tag + r"\s*=\s*(\d+)\s*\(L\s*=\s*(\d+),\s*captured at commit ([0-9a-f]+), ([^)]*)\)", text):
            if int(m.group(2)) == L:
                return int(m.group(1)), "%s: ncu --set full capture at commit %s (%s); not re-measured in this run" % (
                    os.path.relpath(path, ROOT), m.group(3), m.group(4))
    return None, "no committed ncu --set full capture of row %s for L = %d" % (row, L)


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
            su3.su3_expr(z, "01+01*+", [x, y]); su3.su3_expr(z, "01*23*+", [x, y, w, x])        # menu rows of the pipeline
            su3.su3_tune_set(path=3)                                                             # the interpreter
            su3.su3_expr(z, "01+01*+", [x, y]); su3.su3_expr(z, "01*23*+", [x, y, w, x])
            su3.su3_tune_set()
            su3.su3_expr(z, "01*2*3*", [x, y, w, x])                                            # not on the menu
            order.append("%s expr: menu x2, interpreter x3" % name)
            for dim in (0, 3):
                su3.su3_cshift(z, y, dim, 1); su3.su3_mul_shift(z, x, y, dim, 1)                 # bulk-run Cshift, shifted pipeline
            su3.su3_tune_set(path=2)
            su3.su3_cshift(z, y, 0, 1); su3.su3_mul_shift(z, x, y, 1, 1)                         # register kernels
            su3.su3_tune_set(path=3)
            su3.su3_cshift(z, y, 0, 1)                                                           # cp.async gather
            su3.su3_tune_set()
            fb = su3.su3_face_bytes(x, 3, 2)                                                     # (e) faces of a slab: 2 planes
            buf = torch.empty(fb, dtype=torch.uint8, device="cuda")
            su3.su3_face_pack(buf, x, 3, 0, 2); su3.su3_face_unpack(z, buf, 3, L - 2, 2); su3.su3_face_copy(z, 0, x, L - 2, 3, 2)
            psi = su3.su3_vec_wrap(x.desc, w.tensor[:su3.su3_vec_bytes(x.desc)])
            yv_ = su3.su3_vec_wrap(x.desc, z.tensor[:su3.su3_vec_bytes(x.desc)])
            su3.su3_matvec(yv_, x, psi)
        su3.su3_convert(zs, zv)
        for path in (3, 2):                       # the per-thread convert kernels (staged / unstaged), both directions
            su3.su3_tune_set(path=path)
            su3.su3_convert(xv, xs); su3.su3_convert(zs, xv)
        su3.su3_tune_set()
        if prec == su3.SU3_F32:                   # A5 at the long vector lengths of the W sweep (f1)
            for Wl in (16, 32):
                dl = su3.make_desc(L, prec=prec, layout=su3.SU3_VECTOR, W=Wl)
                xl = su3.alloc_field(dl)
                su3.su3_convert(xl, xs); su3.su3_convert(zs, xl)
                del xl
        torch.cuda.synchronize()
        del xs, ys, ws, zs, xv, yv, wv, zv
        torch.cuda.empty_cache()
    print(json.dumps({"profile_pass": True, "L": L, "launches": su3.su3_launch_count() - n0}), flush=True)


def profile_knee(args):
    import torch

    import paper_1710_09409_b200 as su3
    torch.cuda.set_device(0)
    n0 = su3.su3_launch_count()
    for L, prec, W in ((24, su3.SU3_F64, W64), (28, su3.SU3_F32, W32), (32, su3.SU3_F32, W32)):
        dt = torch.float64 if prec == su3.SU3_F64 else torch.float32
        for layout in (su3.SU3_SCALAR, su3.SU3_VECTOR):
            d = su3.make_desc(L, prec=prec, layout=layout, W=W if layout == su3.SU3_VECTOR else 1)
            x, y, z = (su3.alloc_field(d) for _ in range(3))
            x.tensor.view(dt).normal_(); y.tensor.view(dt).normal_()
            for _ in range(3):
                su3.su3_mul(z, x, y)
            torch.cuda.synchronize()
    print(json.dumps({"profile_knee": True, "launches": su3.su3_launch_count() - n0}), flush=True)


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
    if args.profile_pass or args.profile_knee:
        if rank == 0:
            (profile_pass if args.profile_pass else profile_knee)(args)
        return
    if world != args.gpus:
        log("note: --gpus %d but WORLD_SIZE=%d; using WORLD_SIZE (launch N>1 with torch.distributed.run)" % (args.gpus, world))
    r = run_ours(args, rank, world, local_rank)
    torch = r["torch"]
    e2e = None if args.no_e2e else run_e2e(args, r, world)
    halo_leg = None
    if args.halo and world > 1 and r["dist"] is not None and r["dist"].get_backend() == "nccl":
        halo_leg = run_halo(args, r, world, rank)
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
    # Nominal pin-rate peaks, both stated: nvidia-smi's clocks.max.mem (3996 MHz on B200, the figure ncu's
    # dram__throughput is relative to) and the CUDA attribute cudaDevAttrMemoryClockRate (3746 MHz on the same
    # chip); peak = clock x 2 (DDR) x bus width / 8.  `pin_rate_peak` is the nvidia-smi one.
    bus = r["info"]["bus_width_bits"]
    pin_attr = r["info"]["mem_clock_khz"] * 1e3 * 2 * bus / 8 / 1e9
    mem_max = r["clk"].get("mem_max_mhz")
    pin_rate = mem_max * 1e6 * 2 * bus / 8 / 1e9 if mem_max else pin_attr
    traffic, traffic_src = ncu_traffic(args.L)
    roofline = {"bound": "hbm", "kernel": "su3_pipe_kernel<double,W=1,OP_MUL> (row A1, z=x*y fp64 scalar)",
                "achieved": a1["GBps"], "peak": peak, "unit": "GB/s", "frac": a1["GBps"] / peak, "peak_source": peak_src,
                "algorithmic_bytes_per_launch": 3 * B, "avg_launch_ms": a1["ms"],
                "frac_of_same_run_copy": a1["frac_of_copy"], "pin_rate_peak": pin_rate, "frac_of_pin_rate_peak": a1["GBps"] / pin_rate,
                "pin_rate_peak_source": "nvidia-smi clocks.max.mem %s MHz x 2 x %d bit / 8" % (mem_max, bus) if mem_max
                                        else "cudaDevAttrMemoryClockRate x 2 x bus / 8",
                "pin_rate_peak_cuda_attr": pin_attr,
                "pin_rate_peak_cuda_attr_source": "cudaDevAttrMemoryClockRate %.0f MHz x 2 x %d bit / 8" % (r["info"]["mem_clock_khz"] / 1e3, bus),
                "traffic": traffic, "traffic_source": traffic_src,
                "traffic_by_kernel": {row: dict(zip(("traffic", "source"), ncu_traffic(args.L, row)), algorithmic_bytes=nb)
                                      for row, nb in (("A1", 3 * B), ("A5", 2 * B))}}
    cpu = None
    if rank == 0 and not args.no_cpu:
        cpu = run_cpu_baseline(args, r["host"])
    if r["dist"] is not None:
        r["dist"].barrier()
        r["dist"].destroy_process_group()
    if rank != 0:
        return
    line = {
        "metric": METRIC, "value": r["value"], "unit": UNIT, "n_gpus": world, "gpu": r["gpu_name"], "steps": args.steps, "warmup": args.warmup, "warmup_steps_run": r["nwarm"],
        "ms_per_step": r["ms_per_step"], "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
        "dtype": "f64", "data": "synthetic",
        "config": {"workload": "BASELINE.json configs[4] top point: %d^4 lattice per GPU (%d matrices, %.3f GB per field), "
                               "fp64 complex, scalar + vector(W=%d) layouts, rows A1-A6 per step" % (args.L, nmat, B / 1e9, W64),
                   "L": args.L, "step_bytes": r["step_bytes"], "step_flops": r["step_flops"],
                   "l2_policy": "inputs larger than L2 (every launch streams >= %.1f GB; L2 = %.0f MB)" % (2 * B / 1e9, r["info"]["l2_bytes"] / 1e6),
                   "parallelism": "independent x3 slabs, no collective" if world > 1 else "single GPU"},
        "GFLOPps": world * r["step_flops"] / (r["ms_per_step"] * 1e-3) / 1e9,
        "gpu_launches": r["launches"], "clocks": r["clk"], "e2e": e2e, "roofline": roofline, "cpu_baseline": cpu,
        "ops": ops, "ceilings_GBps": {k: v for k, v in ceilings.items() if k not in ("wsweep", "by_size", "convert_f32", "launch_floor_us")},
        "launch_floor_us": ceilings.get("launch_floor_us"),
        "ceilings_by_size": ceilings.get("by_size"), "convert_f32": ceilings.get("convert_f32"),
        "wsweep": ceilings.get("wsweep"), "next_rows": next_rows, "halo": halo_leg, "sweep": sweep, "checks": r["checks"],
        "wall_s_timed_region": r["t_wall"],
        # the paper's own numbers for z = x*y, as context only (other hardware, fp32, volumes unstated)
        "paper_context": {"hardware": "NVIDIA GTX 1080, 288 GB/s peak, ~240 GB/s sustainable (P:156)",
                          "z=x*y scalar AoS layout, CUDA/Jitify, no coalesced_ptr": "~120 GB/s (about half of sustainable)",
                          "z=x*y with coalesced_ptr (AoS -> AoSoAoS)": "saturates the memory bandwidth (~240 GB/s)",
                          "vector layout on GP100/V100": "follows the STREAM triad; plateau only at 16 threads per block (P:199-203)"},
    }
    emit(line)


def _compact(v, digits=6):
    """floats to `digits` significant digits, NaN/inf to None (strict JSON), containers recursively"""
    if isinstance(v, float):
        if v != v or v in (float("inf"), float("-inf")):
            return None
        return float("%.*g" % (digits, v))
    if isinstance(v, dict):
        return {k: _compact(x, digits) for k, x in v.items()}
    if isinstance(v, (list, tuple)):
        return [_compact(x, digits) for x in v]
    return v


HEADLINE_KEYS = ("metric", "value", "unit", "n_gpus", "gpu", "steps", "warmup", "ms_per_step", "higher_is_better", "scaling",
                 "vs_baseline", "dtype", "data", "gpu_launches", "config", "clocks", "checks", "roofline", "cpu_baseline",
                 "e2e", "bar", "GFLOPps", "detail")
HEADLINE_MAX_BYTES = 4096


def headline(line):
    """The record the driver parses: the contract keys, `roofline` (A1, the dominant kernel family, at top level as the
    contract asks; A1 and the largest single kernel A5 side by side under `kernels`), `cpu_baseline`, `e2e` and a digest
    of the north_star bar (z = x*y at 48^4 and 64^4, GB/s and fraction of the same-size copy) -- under 4 KB.  Everything
    else (sweep, ceilings, W sweep, next rows, per-config CPU points, paper context) is the detail record."""
    pick = lambda d, keys: {k: d[k] for k in keys if d is not None and k in d}
    ops = {o["row"]: o for o in line.get("ops") or []}
    roof = line.get("roofline") or {}
    kernels = []
    for row, name, nbytes_key in (("A1", "su3_pipe_kernel<double,1,OP_MUL> z=x*y", "A1"), ("A5", "su3_convert_tma_kernel<double2,4> scalar->vector", "A5")):
        o = next((v for k, v in ops.items() if k.startswith(row)), None)
        if o is None:
            continue
        t = (roof.get("traffic_by_kernel") or {}).get(row) or {}
        kernels.append({"row": row, "kernel": name, "achieved": o["GBps"], "peak": roof.get("peak"),
                        "frac": o["frac_of_measured_peak"], "frac_of_same_run_copy": o["frac_of_copy"],
                        "avg_launch_ms": o["ms"], "algorithmic_bytes_per_launch": t.get("algorithmic_bytes"),
                        "traffic": t.get("traffic"), "traffic_source": t.get("source")})
    roofline = pick(roof, ("bound", "kernel", "achieved", "peak", "unit", "frac", "traffic", "traffic_source", "peak_source",
                           "algorithmic_bytes_per_launch", "avg_launch_ms", "frac_of_same_run_copy", "pin_rate_peak"))
    roofline["kernels"] = kernels
    cpu = line.get("cpu_baseline")
    if cpu is not None:
        cpu = dict(pick(cpu, ("value", "unit", "cores", "kind", "sample", "ms_per_step", "stream_triad_GBps")),
                   one_thread_GBps=(cpu.get("one_thread") or {}).get("GBps"))
    e2e = line.get("e2e")
    if e2e is not None:
        e2e = dict(pick(e2e, ("value", "unit", "h2d_bytes_per_step", "d2h_bytes_per_step", "ms_per_step", "steps", "api",
                              "host_result_matches_device")),
                   host_result_vs_oracle_sampled_ok=(e2e.get("host_result_vs_oracle_sampled") or {}).get("ok"))
    bar = {"%d^4 %s %s" % (p["L"], p["prec"], p["layout"]): [p["GBps"], p.get("frac_of_copy")]
           for p in line.get("sweep") or [] if p.get("L") in (48, 64)}
    head = {k: line.get(k) for k in HEADLINE_KEYS if k in line}
    head.update({"roofline": roofline, "cpu_baseline": cpu, "e2e": e2e,
                 "bar": {"what": "z=x*y: [GB/s, fraction of the same-run same-size copy]; north_star bar 0.85", "points": bar},
                 "detail": "stderr line 'DETAIL {json}' and gpurun_out/bench_detail.json"})
    head = _compact(head)
    for k in head["roofline"]["kernels"] + [head["roofline"]]:     # provenance strings: the profile file says the rest
        if isinstance(k.get("traffic_source"), str) and len(k["traffic_source"]) > 160:
            k["traffic_source"] = k["traffic_source"][:157] + "..."
    if len(json.dumps(head, allow_nan=False)) > HEADLINE_MAX_BYTES:  # never let prose push the record over the limit
        for obj, key in ((head["roofline"], "traffic_source"), (head["roofline"], "peak_source"), (head.get("e2e") or {}, "api"),
                         (head.get("cpu_baseline") or {}, "sample"), (head["config"], "workload")):
            if isinstance(obj.get(key), str) and len(obj[key]) > 120:
                obj[key] = obj[key][:117] + "..."
        for k in head["roofline"]["kernels"]:
            if isinstance(k.get("traffic_source"), str):
                k["traffic_source"] = k["traffic_source"][:80]
    return head


def emit(line):
    """stdout: ONE compact line (the headline record, strict JSON, < 4 KB).  stderr and gpurun_out/: the full record."""
    detail = json.dumps(_compact(line, 9), allow_nan=False)
    print("DETAIL " + detail, file=sys.stderr, flush=True)
    try:
        out = os.path.join(os.path.dirname(os.path.abspath(__file__)), "gpurun_out")
        os.makedirs(out, exist_ok=True)
        with open(os.path.join(out, "bench_detail.json"), "w") as f:
            f.write(detail + "\n")
    except OSError as e:
        log("note: could not write gpurun_out/bench_detail.json: %s" % e)
    print(json.dumps(headline(line), allow_nan=False), flush=True)


if __name__ == "__main__":
    main()
