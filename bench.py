#!/usr/bin/env python
"""bench.py -- throughput of the particle-update hot path on B200 (contract: task prompt, section 4).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--workload c2] [--impl reference]

A "step" is one pass of the whole hot path over one batch of
synthetic input: one C-ABI trace call over all seeds of the workload -- Morton presort, the
persistent advection kernel (fetch, cell location, trilinear gather, RK stages, termination,
vertex record, refill) until every particle has terminated.  Default workload = the LARGEST
single-GPU configuration, BASELINE.json configs[4] (C5): 1024^3 turbulence (12.9 GB), 16,777,216
seeds, DP5(4) tol 1e-5, max 8,000 steps, throughput recording (capacity 64, stride 128; SURVEY.md
8(d) table) -- it stands in for the paper's only benchmark volume (1K^3 voxels).
The same JSON line carries BASELINE.json configs[1] (C2: 256^3, 1,048,576 seeds, RK4 h = 0.25,
max 2,000, capacity 256 stride 8) under "also": {"c2": {...}} with the same fields.

metric  = RK particle-steps per second (step ATTEMPTS), whole job over all ranks.
value   = device-resident inputs, CUDA events on the launching stream around each step.
e2e     = the same through the C-ABI *_host calls with pinned HOST buffers (streamlines: seeds in,
          assembled polylines out -- streami_trace_streamlines_lines_host)
          (H2D of the seeds and D2H of every output inside the timed region).
roofline= the advection kernel alone (event pair recorded by the library around its launch), against
          MEASURED_PEAKS.json hbm_gbs:
          traffic            dram__bytes_read + write per launch, ncu (profiles/traffic.csv, stamped with the
                             commit and kernel time it was captured at; flagged when stale)
          achieved / frac    that measured traffic / LIVE kernel time (/ peak): what the memory system carries
                             (= dram_gbs / dram_frac).  Without a traffic row: the algorithmic rate
          achieved_algorithmic / compulsory_frac
                             ALGORITHMIC bytes = SURVEY.md 8(d)'s compulsory row (what the method must move
                             with perfect caching: 18 / 36 / 72 B per RK4-steady / RK4-unsteady / DP5(4) step
                             attempt + 12 B per stored vertex + 36 B per particle) / live kernel time (/ peak)
          wasted_traffic     traffic / algorithmic bytes
          useful_request_gbs bytes the samples ask for (8 vertices x 12 B per sample and slice), a RATE only:
                             the register cell cache answers most of them without any memory access
          l2                 lts__t_sectors_op_read x 32 B per launch (ncu) / live kernel time against the
                             L2-resident gather ceiling measured on this chip
cpu_baseline = the fp32 oracle, as it stands, on the host cores, on a bounded strided sample.

Multi-GPU (torchrun): the field is replicated, every rank traces its own 1,048,576 seeds
(engine seed 42 + rank), no data-path collective -> "scaling": "weak".
`--impl reference` times the CPU oracle instead (rank 0 only).
"""
import argparse
import json
import os
import subprocess
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

METRIC = "rk_particle_steps_per_sec"
UNIT = "particle-steps/s"

# name -> recipe (throughput-run recording parameters)
WORKLOADS = {
    "c1": dict(kind="abc", N=32, n=1024, ext=None, prm=dict(integrator=0, h=0.01, max_steps=1000,
               vmin=1e-6, capacity=1001, stride=1)),
    "c2": dict(kind="turb", N=256, M=512, kmax=64, n=1 << 20, prm=dict(integrator=0, h=0.25,
               max_steps=2000, vmin=1e-6, capacity=256, stride=8)),
    "c3": dict(kind="bricks", N=512, M=512, kmax=64, n=1 << 22, nb=(2, 2, 2), prm=dict(integrator=0,
               h=0.25, max_steps=4000, vmin=1e-6, capacity=256, stride=16)),
    "c4": dict(kind="gyre", m=4096, nsteps=1000, prm=dict(integrator=0, h=0.05, vmin=1e-6)),
    "c5": dict(kind="turb", N=1024, M=1024, kmax=256, n=1 << 24, prm=dict(integrator=1, h=0.25,
               h_min=0.01, h_max=1.0, atol=1e-5, rtol=1e-5, max_steps=8000, vmin=1e-6, capacity=64,
               stride=128),
               # 137 GB of CELL records: more than the half of the free memory AUTO allows itself, so the
               # caller asks for it (streami.h: STREAMI_LAYOUT_CELL)
               layout=4),
    # pathlines ("easy to implement within the framework"): streamlines through C4's time-sliced
    # field, 1 Mi seeds uniform in the domain (never the reported headline)
    "p4": dict(kind="path", n=1 << 20, prm=dict(integrator=0, h=0.05, max_steps=1000, vmin=1e-7, t0=0.0,
               capacity=64, stride=16)),
    # the paper's other field type: a 128^3 turbulence grid re-expressed as 127^3 hexahedra
    # (PAPER.md:159), bins 127^3, RK4 (never the reported headline)
    "u1": dict(kind="mesh", N=128, M=128, kmax=32, n=1 << 18, nbins=(127, 127, 127), prm=dict(integrator=0, h=0.25,
               max_steps=500, vmin=1e-6, capacity=64, stride=8)),
}
DESCR = {
    "c1": "C1 ABC 32^3, 1,024 seeds, RK4 h=0.01, max 1,000",
    "c2": "C2 turbulence 256^3 (512 modes), 1,048,576 seeds, RK4 h=0.25, max 2,000 steps",
    "c3": "C3 turbulence 512^3 in 2x2x2 bricks (ghost 1), 4,194,304 seeds, RK4 h=0.25, max 4,000",
    "c4": "C4 double gyre 256x128x64 x 64 slices, 4,096-point rake, 1,000 steps, streaklines",
    "c5": "C5 turbulence 1024^3 (1,024 modes), 16,777,216 seeds, DP5(4) tol 1e-5, max 8,000",
    "p4": "P4 pathlines through C4's double gyre (64 slices), 1,048,576 seeds, RK4 h=0.05, max 1,000",
    "u1": "U1 hexahedral mesh: 128^3 turbulence grid as 2,048,383 hexahedra, 262,144 seeds, RK4 h=0.25, max 500",
}


class ClockSampler:
    """nvidia-smi clocks / throttle reasons sampled every 200 ms during the timed region."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, index):
        self.rows, self.proc, self.thr = [], None, None
        try:
            self.proc = subprocess.Popen(
                ["nvidia-smi", "-i", str(index), "--query-gpu=" + self.Q,
                 "--format=csv,noheader,nounits", "-lms", "200"],
                stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.thr = threading.Thread(target=self._read, daemon=True)
            self.thr.start()
        except OSError:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.rows.append((time.time(), line.strip()))

    def stop(self, t0, t1):
        if self.proc is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        time.sleep(0.25)
        self.proc.terminate()
        try:
            self.proc.wait(timeout=5)
        except subprocess.TimeoutExpired:
            self.proc.kill()
        sm, smax, power, reasons = [], None, [], set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for ts, line in self.rows:
            f = [x.strip() for x in line.split(",")]
            if len(f) < 7:
                continue
            try:
                smax = float(f[1])
                if t0 <= ts <= t1 + 0.2:
                    sm.append(float(f[0])); power.append(float(f[2]))
                    for k, nm in enumerate(names):
                        if f[3 + k].lower().startswith("active"):
                            reasons.add(nm)
            except ValueError:
                continue
        sm.sort()
        return {"sm_mhz": sm[len(sm) // 2] if sm else None, "sm_max_mhz": smax,
                "power_w_max": max(power) if power else None, "samples": len(sm),
                "reasons": sorted(reasons)}


def parse_args():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=5)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--workload", default=None, choices=sorted(WORKLOADS),
                    help="default: c5 (the largest single-GPU config) with c2 carried under \"also\"")
    ap.add_argument("--layout", type=int, default=0, help="0 auto, 1 packed3, 2 float4, 3 xpair, 4 cell, 5 xyquad")
    ap.add_argument("--opt", action="append", default=[], help="library option name=value")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--no-cpu", action="store_true", help="skip the cpu_baseline leg")
    ap.add_argument("--cpu-seconds", type=float, default=12.0)
    return ap.parse_args()


# ------------------------------------------------------------------------------------------------
# workloads: device-resident inputs for our arm, host arrays for the oracle legs
# ------------------------------------------------------------------------------------------------
def host_inputs(name, rank, need_field=True):
    """Host-side (numpy) field + seeds of a workload, for the oracle legs.  Large turbulence
    fields are filled on the GPU when one is present (workloads/fill.cu, input generation only)
    and copied back: the oracle then sees the same bytes as the CUDA path."""
    import numpy as np
    import workloads as wl
    w = WORKLOADS[name]
    if w["kind"] == "abc":
        return wl.abc_field(w["N"]), wl.seeds_uniform(shard_seed(rank), w["n"], [2 * np.pi] * 3)
    if w["kind"] == "gyre":
        return wl.double_gyre_field(), wl.rake_c4()
    if w["kind"] == "path":
        return wl.double_gyre_field(), wl.seeds_uniform(shard_seed(rank), w["n"], [2.0, 1.0, 1.0])
    seeds = wl.seeds_uniform(shard_seed(rank), w["n"], [w["N"] - 1.0] * 3)
    fld = None
    if need_field:
        import torch
        if torch.cuda.is_available():
            fld, _ = wl.turb_field_cuda(w["N"], w["M"], 1.0, w["kmax"])
        else:
            if w["N"] > 64:
                raise SystemExit("no GPU: the %d^3 field cannot be generated on the CPU in time" % w["N"])
            fld = wl.turb_field_cpu(w["N"], w["M"], 1.0, w["kmax"])
    return fld, seeds


class Job:
    """One workload on one GPU through the Python binding of the C ABI."""

    def __init__(self, name, rank, layout):
        import numpy as np
        import torch
        import workloads as wl
        import paper_2606_02627_b200 as S
        self.S, self.torch, self.np, self.name = S, torch, np, name
        w = self.w = WORKLOADS[name]
        if layout == 0:
            layout = w.get("layout", 0)
        self.kind = w["kind"]
        self.host_field = None
        if self.kind == "abc":
            fld = self.host_field = wl.abc_field(w["N"])
            self.data = torch.from_numpy(fld.data).cuda()
            self.field = S.streami_field_create(fld.dims, fld.origin, fld.spacing, 1, 1.0, self.data, layout)
            self.seeds_h = wl.seeds_uniform(shard_seed(rank), w["n"], [2 * np.pi] * 3)
        elif self.kind == "gyre":
            fld = self.host_field = wl.double_gyre_field()
            self.data = torch.from_numpy(fld.data).cuda()
            self.field = S.streami_field_create(fld.dims, fld.origin, fld.spacing, fld.nslices,
                                                fld.slice_dt, self.data, layout)
            self.seeds_h = wl.rake_c4()
        elif self.kind == "path":
            fld = self.host_field = wl.double_gyre_field()
            self.data = torch.from_numpy(fld.data).cuda()
            self.field = S.streami_field_create(fld.dims, fld.origin, fld.spacing, fld.nslices,
                                                fld.slice_dt, self.data, layout)
            self.seeds_h = wl.seeds_uniform(shard_seed(rank), w["n"], [2.0, 1.0, 1.0])
        elif self.kind == "mesh":
            N = w["N"]
            fld, dev = wl.turb_field_cuda(N, w["M"], 1.0, w["kmax"], host=True)
            del dev
            self.host_field = fld
            self.mesh_arrays = wl.hexmesh_from_grid(fld.dims, fld.origin, fld.spacing, fld.data[0])
            X, V, H, lo, hi = self.mesh_arrays
            self.field = S.Mesh(X, V, H, lo, hi, w["nbins"])
            self.data = None
            self.seeds_h = wl.seeds_uniform(shard_seed(rank), w["n"], [N - 1.0] * 3)
        else:
            N = w["N"]
            want_host = N <= 512
            fld, dev = wl.turb_field_cuda(N, w["M"], 1.0, w["kmax"], host=want_host)
            self.host_field = fld
            if self.kind == "bricks":
                self.data = wl.cut_bricks_cuda(dev, (N, N, N), w["nb"], 1)
                del dev
                self.field = S.streami_field_create_bricked((N, N, N), (0, 0, 0), (1, 1, 1), w["nb"], 1,
                                                            self.data, layout)
            else:
                self.data = dev
                self.field = S.streami_field_create((N, N, N), (0, 0, 0), (1, 1, 1), 1, 1.0, dev, layout)
            self.seeds_h = wl.seeds_uniform(shard_seed(rank), w["n"], [N - 1.0] * 3)
        self.layout, self.owned_bytes = self.field.info() if self.kind != "mesh" else (0, 224 * self.mesh_arrays[2].shape[0])
        self.n = self.seeds_h.shape[0]
        self.seeds = torch.from_numpy(self.seeds_h).cuda()
        dev = "cuda"
        if self.kind == "gyre":
            self.nsteps = w["nsteps"]
            npart = self.n * self.nsteps
            self.verts = torch.empty((3, self.nsteps, self.n), dtype=torch.float32, device=dev)
            self.counts = torch.empty(self.n, dtype=torch.int32, device=dev)
        else:
            npart = self.n
            cap = w["prm"]["capacity"]
            self.verts = torch.empty((3, self.n, cap), dtype=torch.float32, device=dev)
            self.counts = torch.empty(self.n, dtype=torch.int32, device=dev)
        self.npart = npart
        self.steps_o = torch.empty(npart, dtype=torch.int32, device=dev)
        self.status_o = torch.empty(npart, dtype=torch.int32, device=dev)
        self.final_o = None if self.kind == "gyre" else torch.empty((3, self.n), dtype=torch.float32, device=dev)
        self.totals_o = torch.zeros(4, dtype=torch.int64, device=dev)
        self.prm = S.params(out_steps=self.steps_o, out_status=self.status_o, out_final=self.final_o,
                            out_totals=self.totals_o, **w["prm"])
        self.nrounds = 0
        # pinned host buffers for the e2e leg
        self.h = None

    # -- one step, inputs and outputs resident in HBM ------------------------------------------
    def step_device(self):
        S = self.S
        if self.kind == "mesh":
            S.streami_mesh_trace_streamlines(self.field, self.seeds, self.prm, self.verts, self.counts)
        elif self.kind == "gyre":
            S.streami_trace_streaklines(self.field, self.seeds, self.nsteps, self.prm, self.verts, self.counts)
        elif self.kind == "bricks":
            self.nrounds, _ = S.streami_brick_advect(self.field, self.seeds, self.prm, self.verts, self.counts)
        else:
            S.streami_trace_streamlines(self.field, self.seeds, self.prm, self.verts, self.counts)

    # -- one step through host buffers -----------------------------------------------------------
    def _pinned(self):
        t = self.torch
        if self.h is None:
            pin = lambda x: t.empty(x.shape, dtype=x.dtype).pin_memory()
            self.h = dict(seeds=t.from_numpy(self.seeds_h).pin_memory(), verts=pin(self.verts),
                          counts=pin(self.counts), steps=pin(self.steps_o), status=pin(self.status_o),
                          final=None if self.final_o is None else pin(self.final_o),
                          totals=t.zeros(4, dtype=t.int64).pin_memory())
            if self.kind != "gyre":
                # polyline buffers instead of the capacity-padded slot array
                self.h["verts"] = None; self.h["counts"] = None
                self.h["offsets"] = t.zeros(self.n + 1, dtype=t.int64).pin_memory()
                self.h["points"] = t.empty((self.n * self.w["prm"]["capacity"], 3), dtype=t.float32).pin_memory()
                self.e2e_points = 0
            kw = dict(self.w["prm"])
            self.prm_h = self.S.params(out_steps=None, out_status=None, out_final=None, out_totals=None, **kw)
            self.prm_h.out_steps = self.h["steps"].data_ptr()
            self.prm_h.out_status = self.h["status"].data_ptr()
            if self.h["final"] is not None:
                self.prm_h.out_final = self.h["final"].data_ptr()
            self.prm_h.out_totals = self.h["totals"].data_ptr()
        return self.h

    def e2e_bytes(self):
        h = self._pinned()
        nb = lambda x: 0 if x is None else x.numel() * x.element_size()
        bi = nb(h["seeds"])
        bo = sum(nb(h[k]) for k in ("verts", "counts", "steps", "status", "final", "totals"))
        if self.kind != "gyre":                        # offsets + the points actually delivered
            bo += nb(h["offsets"]) + 12 * int(self.e2e_points)
        return bi, bo

    def step_host(self):
        """One step through the C-ABI host-buffer calls: H2D of the seeds / rake points, the
        trace, D2H of every output, stream sync -- all inside the library."""
        h, S = self._pinned(), self.S
        if self.kind == "mesh":
            self.e2e_points, _ = S.streami_mesh_trace_streamlines_lines_host(self.field, h["seeds"], self.prm_h,
                                                                             h["offsets"], h["points"])
        elif self.kind == "gyre":
            S.streami_trace_streaklines_host(self.field, h["seeds"], self.nsteps, self.prm_h, h["verts"], h["counts"])
        else:
            # streamlines: the host application's end product is the assembled polylines (the paper's
            # getLines): offsets + points; only stored vertices cross the bus
            self.e2e_points, _ = S.streami_trace_streamlines_lines_host(self.field, h["seeds"], self.prm_h,
                                                                        h["offsets"], h["points"])

    def host_field_lazy(self):
        """The field on the host for the oracle legs.  The 1024^3 field (12.9 GB) is copied back only when
        asked for: the same bytes the CUDA path traced."""
        if self.host_field is None and self.kind == "turb" and self.data is not None:
            import workloads as wl
            N = self.w["N"]
            self.host_field = wl.Field((N, N, N), (0.0, 0.0, 0.0), (1.0, 1.0, 1.0), self.data.cpu().numpy())
        return self.host_field

    def release_pinned(self):
        self.h = None

    def close(self):
        """Free the field handle and every device buffer of this job (the next workload needs the memory)."""
        if self.kind != "mesh":
            self.field.destroy()
        else:
            self.field.destroy()
        for k in ("data", "seeds", "verts", "counts", "steps_o", "status_o", "final_o", "totals_o", "prm", "h", "host_field"):
            setattr(self, k, None)

    def work(self):
        """(attempted steps, accepted steps, field samples, hand-offs, stored vertices) of the
        last device step."""
        tot = [int(x) for x in self.totals_o.cpu().tolist()]
        stored = self.npart if self.kind == "gyre" else int(self.counts.to(self.torch.int64).sum().item())
        return tot[0], tot[1], tot[2], tot[3], stored


# ------------------------------------------------------------------------------------------------
# the oracle legs (cpu_baseline and --impl reference): the only places that execute oracle/
# ------------------------------------------------------------------------------------------------
class OracleRun:
    """The fp32 CPU oracle, as it stands, on a strided sample of the workload's particles."""

    def __init__(self, name, fld, seeds):
        import oracle
        import workloads as wl
        self.o, self.name, self.w = oracle, name, WORKLOADS[name]
        self.kind = self.w["kind"]
        self.seeds = seeds
        oracle.build()
        prm = dict(self.w["prm"])
        time_mode = prm.pop("time_mode", 0)
        if self.kind == "gyre":
            prm.update(capacity=1, stride=1, max_steps=self.w["nsteps"])
        self.prm = oracle.params(**prm)
        if self.kind == "mesh":
            X, V, H, lo, hi = wl.hexmesh_from_grid(fld.dims, fld.origin, fld.spacing, fld.data[0])
            self.field = oracle.HexMesh(X, V, H, lo, hi, self.w["nbins"])
        elif self.kind == "bricks":
            N = self.w["N"]
            boxes = wl.brick_boxes(fld.dims, self.w["nb"], 1)
            cut = wl.cut_bricks(fld, self.w["nb"], 1)
            self.field = [oracle.grid(c, None, fld.origin, fld.spacing, gdims=fld.dims, lo=lo, hi=hi)
                          for c, (lo, hi) in zip(cut, boxes)]
        else:
            self.field = oracle.grid(fld.data, fld.dims, fld.origin, fld.spacing, fld.nslices, fld.slice_dt, time_mode)
        self.cores = oracle.num_threads()

    def run(self, stride):
        """Trace every stride-th particle; returns (attempted steps, seconds, particles)."""
        o = self.o
        sub = self.seeds[::stride]
        t0 = time.perf_counter()
        if self.kind == "mesh":
            r = o.hexmesh_streamlines(self.field, sub, self.prm, "f32", record=False)
        elif self.kind == "gyre":
            r = o.streaklines(self.field, sub, self.w["nsteps"], self.prm, "f32")
        elif self.kind == "bricks":
            r = o.brick_advect(self.field, self.w["nb"], sub, self.prm, "f32", record=False)
        else:
            r = o.streamlines(self.field, sub, self.prm, "f32", record=False)
        dt = time.perf_counter() - t0
        npart = sub.shape[0] * (self.w["nsteps"] if self.kind == "gyre" else 1)
        return int(r.totals[0]), dt, npart

    def bounded(self, seconds):
        """Pick the stride so that one run takes about `seconds` (probe first), then run it."""
        n = self.seeds.shape[0]
        probe = max(1, n // max(64, 16 * self.cores))
        a, dt, _ = self.run(probe)
        rate = a / max(dt, 1e-6)
        per_particle = max(a, 1) / max(1, len(range(0, n, probe)))
        want = max(1.0, rate * seconds / per_particle)
        stride = max(1, int(n / want))
        a, dt, npart = self.run(stride)
        for _ in range(2):                      # the probe under-uses the cores: re-aim if far off
            if dt >= 0.4 * seconds or stride == 1:
                break
            stride = max(1, int(stride * dt / seconds))
            a, dt, npart = self.run(stride)
        return a, dt, npart, stride


def reference_arm(args, rank):
    """--impl reference: the oracle on the host cores; each step = one bounded sample."""
    if rank != 0:
        return
    fld, seeds = host_inputs(args.workload, 0)
    orc = OracleRun(args.workload, fld, seeds)
    per_step = max(2.0, min(30.0, 150.0 / max(1, args.steps + args.warmup)))
    a, dt, npart, stride = orc.bounded(per_step)
    for _ in range(max(0, args.warmup - 1)):
        orc.run(stride)
    tot_a, tot_t = 0, 0.0
    for _ in range(args.steps):
        a, dt, npart = orc.run(stride)
        tot_a += a; tot_t += dt
    value = tot_a / tot_t
    sample = "every %d-th particle (%d particles, %d step attempts per step)" % (stride, npart, tot_a // max(1, args.steps))
    print(json.dumps({
        "impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus,
        "steps": args.steps, "warmup": args.warmup, "ms_per_step": 1e3 * tot_t / args.steps,
        "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f32",
        "data": "synthetic", "config": {"workload": DESCR[args.workload], "sample": sample},
        "cpu_baseline": {"value": value, "unit": UNIT, "cores": orc.cores, "kind": "oracle", "sample": sample},
        "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0}))


# ------------------------------------------------------------------------------------------------
def shard_seed(rank):
    """Seeds are sharded over ranks with no data-path collective: rank r draws its own
    `seeds_per_gpu` seeds from engine seed 42 + r (rank 0 = BASELINE.json's seed 42); the field is
    replicated.  Weak scaling: per-GPU work is fixed as N grows."""
    return 42 + rank


class Reducer:
    """The only cross-rank traffic of the bench: a barrier, MAX of the timed region and SUM of the
    work counters (torch.distributed; NCCL on GPUs, gloo in the CPU tests)."""

    def __init__(self, world, device):
        self.world, self.device = world, device

    def barrier(self):
        import torch
        if self.world > 1:
            import torch.distributed as dist
            dist.barrier()
        if self.device == "cuda":
            torch.cuda.synchronize()

    def _reduce(self, x, op):
        if self.world == 1:
            return x
        import torch
        import torch.distributed as dist
        t = torch.tensor([x], dtype=torch.float64, device=self.device)
        dist.all_reduce(t, op=op)
        return float(t.item())

    def max(self, x):
        import torch.distributed as dist
        return self._reduce(x, dist.ReduceOp.MAX)

    def sum(self, x):
        import torch.distributed as dist
        return self._reduce(x, dist.ReduceOp.SUM)


def job_value(attempts_this_rank, steps, ms_this_rank, red):
    """Whole-job metric: attempts summed over ranks x steps / MAX over ranks of the timed region."""
    total_ms = red.max(ms_this_rank)
    job_attempts = red.sum(float(attempts_this_rank))
    return job_attempts * steps / (total_ms * 1e-3), total_ms, job_attempts


def peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        with open(p) as f:
            return float(json.load(f)["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)"
    return 6650.0, "fallback (B200_PROFILING.md)"


# L2-resident gather ceiling of this chip: random aligned 32-byte reads inside a 48 MB buffer, one per thread and
# iteration, 64 warps per SM (round-1 probe: 8,170 GB/s; 64-byte pieces 8,350).  No driver
# file records an L2 peak, so this measured figure is the denominator of roofline.l2.
L2_GATHER_GBS = 8170.0

# SURVEY.md 8(d), "Compulsory new data (perfect caching)": bytes per step attempt
COMPULSORY_B = {"rk4_steady": 18.0, "rk4_unsteady": 36.0, "dp5": 72.0}


def traffic_row(workload, layout_name):
    """ncu counters of the dominant kernel, per launch (profiles/traffic.csv; profiles/traffic.md says how)."""
    tpath = os.path.join(ROOT, "profiles", "traffic.csv")
    if not os.path.exists(tpath):
        return None
    import csv
    best = None
    with open(tpath) as f:
        for row in csv.DictReader(f):
            if row["workload"] == workload and row.get("layout", layout_name) in (layout_name, ""):
                best = row
    return best


def roofline_of(job, workload, samples, stored, attempts, kern_ms, kern_n, steps, total_ms, world, lay):
    peak, peak_src = peaks()
    launches_per_step = max(1, kern_n // max(1, steps))
    kms = kern_ms / max(1, kern_n)                                   # live, CUDA events on the launching stream
    unsteady = job.kind in ("gyre", "path") and not job.w["prm"].get("time_mode")
    per_attempt = COMPULSORY_B["dp5"] if job.w["prm"].get("integrator") == 1 else (
        COMPULSORY_B["rk4_unsteady"] if unsteady else COMPULSORY_B["rk4_steady"])
    alg = attempts * per_attempt + stored * 12.0 + job.npart * 36.0      # per step (all launches of it)
    useful = samples * (192.0 if unsteady else 96.0) + stored * 12.0 + job.npart * 36.0
    sec = kms * 1e-3
    achieved = (alg / launches_per_step) / sec / 1e9 if kms > 0 else None
    r = {"bound": "hbm", "achieved": achieved, "peak": peak, "unit": "GB/s",
         "frac": None if achieved is None else achieved / peak, "traffic": None,
         "frac_basis": "algorithmic (compulsory) bytes / live kernel time / peak: no ncu traffic row for this workload and layout",
         "achieved_algorithmic": achieved,
         "kernel": {"gyre": "streak_kernel", "mesh": "mesh_trace_kernel"}.get(job.kind, "trace_kernel"),
         "kernel_ms_per_launch": kms, "kernel_launches_per_step": launches_per_step,
         "algorithmic_bytes_per_launch": alg / launches_per_step,
         "algorithmic_basis": "SURVEY.md 8(d) compulsory row: %g B per step attempt + 12 B per stored vertex + 36 B per particle"
                              % per_attempt,
         "compulsory_frac": None if achieved is None else achieved / peak,
         "useful_request_gbs": (useful / launches_per_step) / sec / 1e9 if kms > 0 else None,
         "peak_source": peak_src,
         "kernel_share_of_step": kern_ms / total_ms if world == 1 else None}
    row = traffic_row(workload, lay)
    if row is not None and kms > 0:
        tr = float(row["dram_bytes_per_launch"])
        r["traffic"] = tr
        r["traffic_source"] = row["source"]
        r["dram_gbs"] = tr / sec / 1e9
        r["dram_frac"] = r["dram_gbs"] / peak
        # the headline fraction is what the memory system CARRIES -- measured DRAM bytes per launch
        # (ncu) over the live kernel time over the measured copy peak; the algorithmic (compulsory-bytes) fraction stays
        # beside it as compulsory_frac, and wasted_traffic says how far apart the two are
        r["achieved"] = r["dram_gbs"]; r["frac"] = r["dram_frac"]
        r["frac_basis"] = ("measured DRAM traffic per launch (ncu dram__bytes_read + write, profiles/traffic.csv) / live kernel time "
                           "/ peak; compulsory_frac = SURVEY.md 8(d) compulsory bytes on the same time and peak")
        r["wasted_traffic"] = tr / (alg / launches_per_step)
        cap_ms = float(row["kernel_ms_at_capture"])
        r["traffic_captured_at"] = {"commit": row["commit"], "kernel_ms": cap_ms}
        # the counted bytes belong to the kernel as it was when ncu saw it: flag them when the live kernel has moved
        # (one captured launch cannot be compared with the mean of several launches of different work: C4's windows)
        r["traffic_stale"] = (abs(kms - cap_ms) > 0.10 * cap_ms) if launches_per_step == 1 else None
        lts = float(row["lts_read_bytes_per_launch"])
        r["l2"] = {"achieved": lts / sec / 1e9, "peak": L2_GATHER_GBS, "unit": "GB/s",
                   "frac": lts / sec / 1e9 / L2_GATHER_GBS,
                   "peak_source": "measured on B200: random 32-byte gathers inside an L2-resident 48 MB buffer (DESIGN.md section 6)",
                   "numerator": "lts__t_sectors_op_read.sum x 32 B per launch (ncu) / live kernel time"}
        r["ncu"] = {k: float(row[k]) for k in ("l1_hit_pct", "l2_hit_pct", "active_lanes_per_warp_instruction",
                                               "issue_slots_busy_pct") if row.get(k)}
    return r


def run_workload(name, args, rank, local, world, red, cpu_seconds, steps, warmup):
    """One workload through all legs: device-resident timed region, e2e, roofline, cpu_baseline."""
    import torch
    import paper_2606_02627_b200 as S
    barrier, allmax = red.barrier, red.max
    job = Job(name, rank, args.layout)
    flush = torch.empty(256 << 20, dtype=torch.uint8, device="cuda")     # > 126 MB L2

    for _ in range(warmup):
        job.step_device()
    torch.cuda.synchronize()
    attempts, accepted, samples, handoffs, stored = job.work()

    # ---- timed region: exactly K steps, device-resident ---------------------------------------
    S.streami_set_option("kernel_timing", 1)
    S.streami_kernel_time()
    ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(steps)]
    sampler = ClockSampler(local) if rank == 0 else None
    barrier()
    l0 = S.streami_launch_count()
    t0 = time.time()
    for a, b in ev:
        flush.zero_()                       # L2 flush between timed iterations (outside the events)
        a.record()
        job.step_device()
        b.record()
    barrier()
    t1 = time.time()
    launches = S.streami_launch_count() - l0
    clocks = sampler.stop(t0, t1) if sampler else None
    kern_ms, kern_n = S.streami_kernel_time()
    S.streami_set_option("kernel_timing", 0)
    value, total_ms, job_attempts = job_value(attempts, steps, sum(a.elapsed_time(b) for a, b in ev), red)

    # ---- e2e: host buffers, copies inside the timed region --------------------------------------
    e2e = None
    if not args.no_e2e:
        job.step_host()
        bi, bo = job.e2e_bytes()
        barrier()
        w0 = time.perf_counter()
        for _ in range(steps):
            job.step_host()
        torch.cuda.synchronize()
        w1 = time.perf_counter()
        e_ms = allmax((w1 - w0) * 1e3)
        e2e = {"value": job_attempts * steps / (e_ms * 1e-3), "unit": UNIT,
               "h2d_bytes_per_step": bi, "d2h_bytes_per_step": bo, "ms_per_step": e_ms / steps}
        job.release_pinned()
        barrier()
    del flush

    lay = {1: "packed3", 2: "float4", 3: "xpair", 4: "cell", 5: "xyquad"}.get(job.layout, str(job.layout))
    if job.kind == "mesh":
        lay = "224-byte cell records (8 corner positions + 8 corner values + box)"
    out = None
    if rank == 0:
        roofline = roofline_of(job, name, samples, stored, attempts, kern_ms, kern_n, steps, total_ms, world, lay)
        cpu = None
        if world == 1 and not args.no_cpu:
            fld = job.host_field_lazy()
            if fld is not None:
                orc = OracleRun(name, fld, job.seeds_h)
                a, dt, npart, stride = orc.bounded(cpu_seconds)
                cpu = {"value": a / dt, "unit": UNIT, "cores": orc.cores, "kind": "oracle",
                       "sample": "every %d-th particle of the same workload (%d particles, %d step attempts, %.1f s)"
                                 % (stride, npart, a, dt)}
                del orc
        out = {
            "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": steps,
            "warmup": warmup, "ms_per_step": total_ms / steps, "higher_is_better": True,
            "scaling": "weak", "vs_baseline": None, "dtype": "f32", "data": "synthetic",
            "config": {"workload": DESCR[name], "seeds_per_gpu": job.n,
                       "recording": {k: job.w["prm"][k] for k in ("capacity", "stride") if k in job.w["prm"]},
                       "field_layout": lay, "field_bytes_owned": job.owned_bytes,
                       "l2": "flushed between timed steps (256 MiB memset) and the field is larger than L2",
                       "parallelism": "seeds sharded over %d GPU(s), field replicated" % world,
                       "options": {k: S.streami_get_option(k) for k in ("cell_cache", "presort")}},
            "work_per_step_per_gpu": {"step_attempts": attempts, "accepted_steps": accepted,
                                      "field_samples": samples, "handoffs": handoffs,
                                      "stored_vertices": stored, "rounds": job.nrounds},
            "clocks": clocks, "e2e": e2e, "gpu_launches": int(launches), "roofline": roofline,
            "cpu_baseline": cpu,
        }
        if cpu is not None:
            out["vs_cpu_baseline"] = value / cpu["value"]     # context only; vs_baseline stays null (no published number)
    job.close()
    del job
    torch.cuda.empty_cache()
    return out


def main():
    args = parse_args()
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    headline = args.workload or "c5"
    if args.impl == "reference":
        args.workload = headline
        reference_arm(args, rank)
        return
    import torch
    import torch.distributed as dist
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: there is no CPU fallback")
    torch.cuda.set_device(local)
    if world > 1:
        os.environ.setdefault("MASTER_ADDR", "127.0.0.1")
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))
    red = Reducer(world, "cuda")

    import paper_2606_02627_b200 as S
    for kv in args.opt:
        k, v = kv.split("=")
        S.streami_set_option(k, int(v))

    out = run_workload(headline, args, rank, local, world, red, args.cpu_seconds, args.steps, args.warmup)
    if args.workload is None:
        # the default run also carries BASELINE.json configs[1] (C2), the config the metric was first quoted on
        c2 = run_workload("c2", args, rank, local, world, red, min(args.cpu_seconds, 6.0), args.steps, args.warmup)
        if rank == 0:
            out["also"] = {"c2": c2}
            out["gpu_launches"] += c2["gpu_launches"]
            out["config"]["also"] = "c2 = " + DESCR["c2"]
    if rank == 0:
        print(json.dumps(out))
    if world > 1:
        dist.destroy_process_group()


if __name__ == "__main__":
    main()
