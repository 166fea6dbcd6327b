"""bench.py -- smear-step throughput of the lqx library on N B200s (one process per GPU).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--workload c4|c3] [--no-extras]
    python bench.py --impl reference ...        # the CPU oracle on a bounded sample of the same workload
    python bench.py --kernel-only               # timed device region only: the command ncu wraps for the smear kernel
    python bench.py --extras-only               # per-kernel rows of configs 1, 2, 3, 5, Jacobi routine, run-time expressions
    python bench.py --sweep-geometry            # P(N_threads, N_site) of the Jacobi step (the paper's Figs. 1-2)

One "step" = one pass of the whole hot path over the link field: a fused staple-sum smearing step
(alpha = 0.5, all four directions, plaquette of its input accumulated in the same pass) -- K steps
are iterated on ping-pong buffers and the plaquette after the last step gets its own pass, exactly
what lqx_smear_iterate does (BASELINE.json configs[3]: 48^3x96, fp32, near-unit SU(3), plaquette
after each step).  Prints ONE JSON line (rank 0).  The path does not shard (replicas
only): with N > 1 every rank runs an independent replica, value = N * V * K / max-over-ranks time.
"""
from __future__ import annotations

import argparse
import json
import os
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

ALPHA = 0.5
# per site-update -- algorithmic bytes (read 72 + write 72 reals), canonical
# flops of the literal 48-product evaluation, and FMA lane-ops the kernel variants execute
SMEAR_REALS_PER_SITE = 144
SMEAR_CANONICAL_FLOPS = 10080
SMEAR_LANE_OPS = {"literal": 5328, "shared": 4032}
SMEAR_LANE_OPS_LITERAL = SMEAR_LANE_OPS["literal"]  # the algorithmic FMA lane-ops of one site update
PLAQ_REALS_PER_SITE = 72
WORKLOADS = {
    "c4": dict(cfg="c4", recipe="near_unit", desc="BASELINE configs[3]: 48^3x96 fp32 near-unit SU(3) (exp(0.1iH) reunitarised), "
               "iterated smear steps a=0.5, plaquette after each"),
    "c3": dict(cfg="c3", recipe="haar", desc="BASELINE configs[2]: 32^3x64 fp64 Haar SU(3), smear steps a=0.5 + plaquette"),
    # only with --kernel-only --only hop: the lattice of BASELINE configs[1] (16^3x32 fp32), for the ncu capture of k_hop
    "c2": dict(cfg="c2", recipe="haar", desc="BASELINE configs[1]: 16^3x32 fp32 Haar SU(3) + Gaussian fermion, hop"),
}


def _peaks():
    path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(path):
        with open(path) as f:
            p = json.load(f)
        return float(p["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)", float(p.get("sm_max_mhz", 1965.0))
    return 6650.0, "fallback (B200_PROFILING.md 6.65 TB/s)", 1965.0


def _ncu_capture(kernel_name, prec="f32"):
    """Figures of the newest committed ncu capture OF THIS KERNEL: the profiles/r*.md file (newest round letter last)
    whose `Kernel Name` row names `kernel_name`.  Returns (dict of metric -> value in base units, file) or
    (None, reason).  bench.py never runs under ncu; these are recorded figures, used for `traffic` and for naming
    the busiest unit -- a capture of another kernel is never attached to this line."""
    import glob
    import re

    for path in sorted(glob.glob(os.path.join(ROOT, "profiles", "r*.md")), reverse=True):
        text = open(path).read()
        m = re.search(r"^\|\s*Kernel Name\s*\|[^|]*\|(.*)\|\s*$", text, re.M)
        if not m or not re.search(r"\b" + re.escape(kernel_name) + r"\b", m.group(1)):
            continue
        if ("<double" in m.group(1) and prec == "f32") or ("<float" in m.group(1) and prec == "f64"):
            continue  # the other precision's instantiation of this kernel
        vals = {}
        for line in text.splitlines():
            mm = re.match(r"\|\s*([a-z0-9_.]+)\s*\|\s*([\w/%]*)\s*\|(.*)\|\s*$", line)
            if not mm:
                continue
            cols = [c.strip() for c in mm.group(3).split("|")]
            try:
                x = float(cols[-1])
            except ValueError:
                continue
            vals[mm.group(1)] = x * {"Gbyte": 1e9, "Mbyte": 1e6, "Kbyte": 1e3}.get(mm.group(2), 1.0)
        if "dram__bytes_read.sum" in vals and "dram__bytes_write.sum" in vals:
            return vals, "profiles/" + os.path.basename(path)
    return None, f"no committed ncu capture of {kernel_name} under profiles/"


class ClockSampler(threading.Thread):
    """Polls SM clock and throttle reasons through NVML while the timed region runs."""

    def __init__(self, index: int, period_s: float = 0.004):
        super().__init__(daemon=True)
        self.index, self.period = index, period_s
        self.samples, self.reasons = [], set()
        self.max_mhz = None
        self._stop_evt = threading.Event()
        try:
            import pynvml

            pynvml.nvmlInit()
            self.nv = pynvml
            self.h = pynvml.nvmlDeviceGetHandleByIndex(index)
            self.max_mhz = int(pynvml.nvmlDeviceGetMaxClockInfo(self.h, pynvml.NVML_CLOCK_SM))
        except Exception:
            self.nv = None

    def run(self):
        if self.nv is None:
            return
        nv = self.nv
        names = {
            getattr(nv, "nvmlClocksEventReasonHwSlowdown", 0x8): "hw_slowdown",
            getattr(nv, "nvmlClocksEventReasonHwThermalSlowdown", 0x40): "hw_thermal_slowdown",
            getattr(nv, "nvmlClocksEventReasonSwThermalSlowdown", 0x20): "sw_thermal_slowdown",
            getattr(nv, "nvmlClocksEventReasonSwPowerCap", 0x4): "sw_power_cap",
        }
        while not self._stop_evt.is_set():
            try:
                self.samples.append(int(nv.nvmlDeviceGetClockInfo(self.h, nv.NVML_CLOCK_SM)))
                try:
                    r = int(nv.nvmlDeviceGetCurrentClocksEventReasons(self.h))
                except Exception:
                    r = int(nv.nvmlDeviceGetCurrentClocksThrottleReasons(self.h))
                for bit, name in names.items():
                    if r & bit:
                        self.reasons.add(name)
            except Exception:
                pass
            time.sleep(self.period)

    def stop(self):
        self._stop_evt.set()
        self.join(timeout=2.0)
        s = sorted(self.samples)
        return {"sm_mhz": (s[len(s) // 2] if s else None), "sm_max_mhz": self.max_mhz,
                "reasons": sorted(self.reasons), "samples": len(s)}


def _dist(backend="nccl"):
    """(rank, world, local_rank, barrier_fn, max_fn) -- torch.distributed only when launched by torchrun.
    The path does not shard: the group is used for the barrier and the max over ranks
    only.  backend "gloo" is what the CPU tests use (world_size 2, no GPU)."""
    world = int(os.environ.get("WORLD_SIZE", "1"))
    if world <= 1:
        return 0, 1, 0, (lambda: None), (lambda x: x)
    import torch
    import torch.distributed as dist

    rank, local = int(os.environ["RANK"]), int(os.environ.get("LOCAL_RANK", "0"))
    if backend == "nccl":
        torch.cuda.set_device(local)
        dist.init_process_group(backend="nccl", device_id=torch.device(f"cuda:{local}"))
        dev = f"cuda:{local}"
    else:
        dist.init_process_group(backend=backend)
        dev = "cpu"

    def vmax(x):
        t = torch.tensor([float(x)], dtype=torch.float64, device=dev)
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
        return float(t.item())

    return rank, world, local, dist.barrier, vmax


def replica_value(world, sites, steps, ms_max):
    """Whole-job throughput of N independent replicas: every rank updates `sites` sites `steps` times and
    the job takes as long as its slowest rank."""
    return world * sites * steps / (ms_max * 1e-3)


def _gen_links(lat, lqx, li, cfgname, recipe, prec, keep_host=False):
    """Seeded synthetic link field generated with torch on the GPU (input generator only), converted
    AoS -> SoA by the library.  Returns (fields, pinned host copies or None)."""
    import torch

    cfg = li.CONFIGS[cfgname]
    dev = f"cuda:{lat.device}"
    fields, host = [], []
    v = lat.volume
    for mu in range(4):
        if recipe == "haar":
            z = li.haar_su3_complex(cfg["seed"], mu, v, dev)
        else:
            z = li.near_unit_su3_complex(cfg["seed"], mu, v, 0.1, dev)
        a = li._as_real(z, prec)
        del z
        f = lat.alloc(lqx.COLORMAT, lqx.F32 if prec == "f32" else lqx.F64)
        f.import_dev(a)
        torch.cuda.synchronize()
        if keep_host:
            h = torch.empty(a.shape, dtype=a.dtype, pin_memory=True)
            h.copy_(a)
            host.append(h)
        del a
        fields.append(f)
    torch.cuda.empty_cache()
    return fields, (host if keep_host else None)


def _cpu_baseline(orc, dims, prec, host_links, target_s=12.0):
    """The oracle as it stands (native-precision instantiation, OpenMP over its site loop) on a bounded
    sample of the same workload: smear_links for all four directions + the plaquette integrand on the
    first n sites of the full-size host field."""
    import numpy as np

    variant = orc.native_variant(prec)
    u = [h.numpy() if hasattr(h, "numpy") else h for h in host_links]
    v = u[0].shape[0]

    def run(nsites):
        sites = np.repeat(np.arange(nsites, dtype=np.int64), 4)
        mus = np.tile(np.arange(4, dtype=np.int32), nsites)
        t0 = time.perf_counter()
        orc.smear_links(dims, u, ALPHA, sites, mus, variant)
        orc.plaquette_sites(dims, u, np.arange(nsites, dtype=np.int64), variant)
        return time.perf_counter() - t0

    n0 = min(v, 20000)
    run(min(v, 2000))  # page in / spin up the thread pool
    t = run(n0)
    n = int(min(v, max(n0, n0 * target_s / max(t, 1e-6))))
    t = run(n)
    passes = 1
    while n == v and t < 0.75 * target_s:  # the whole field is a few seconds of CPU work: time several whole steps
        t += run(n)
        passes += 1
    out = {"value": passes * n / t, "unit": "site-updates/s", "cores": orc.num_threads(), "kind": "oracle",
           "sample": f"{passes} pass(es) over the first {n} of {v} sites of the full-size field (all 4 directions + "
                     f"plaquette), oracle variant {variant}, {t:.1f} s"}
    # SURVEY 8(d) timing protocol: also ONE host thread, on a sample a tenth of the all-core budget
    nthreads = orc.num_threads()
    try:
        orc.set_num_threads(1)
        n1 = int(min(v, max(2000, out["value"] / max(nthreads, 1) * target_s * 0.25)))
        t1 = run(n1)
        out["single_thread"] = {"value": n1 / t1, "unit": "site-updates/s", "cores": 1,
                                "sample": f"the first {n1} sites, {t1:.1f} s"}
    finally:
        orc.set_num_threads(nthreads)
    return out


def _time_kernel(torch, fn, reps, flush=None):
    """Median and best device time (ms) of fn() over reps launches, CUDA events on the current stream."""
    times = []
    for _ in range(reps):
        if flush is not None:
            flush.add_(1)
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record()
        fn()
        e1.record()
        e1.synchronize()
        times.append(e0.elapsed_time(e1))
    times.sort()
    return times[len(times) // 2], times[0]


def jacobi_listing(lqx, chi, u, kappa, iters, no_smear_dir, norm, work, fused):
    """The paper's Listing 1 as USER code on top of the run-time expression path, the way a
    QDP++ program would state it.  fused = False: literally the listing, one expression per line -- E0 copies,
    E1 for the first direction, E2 ('+=') for the others, E3, E4 (six kernels per iteration).  fused = True:
    one expression per iteration, chi' = s_0 + kappa * sum_mu (...), the iterate ping-ponging between chi and psi
    (no copy).  work = (s_0, psi, h_smear) scratch fields."""
    s0, psi, h = work
    L = lqx.Expr.leaf
    lqx.expr_eval(s0, L(chi))                                             # s_0 = chi

    def hop_terms(f):
        return [L(u[mu]) * lqx.shifted(f, lqx.FORWARD, mu) + lqx.shifted(lqx.adj(u[mu]) * L(f), lqx.BACKWARD, mu)
                for mu in range(4) if mu != no_smear_dir]

    if fused:
        # E0 (psi = chi) disappears too: the iterate ping-pongs between chi and psi, E4 reads whichever holds it
        cur, nxt = chi, psi
        for _ in range(iters):
            terms = hop_terms(cur)
            e = terms[0]
            for t in terms[1:]:
                e = e + t
            lqx.expr_eval(nxt, L(s0) + kappa * e)                         # E1..E3 in one kernel
            cur, nxt = nxt, cur
        lqx.expr_eval(chi, (1.0 / norm) * L(cur))                         # chi = iterate / norm (E4)
        return
    for _ in range(iters):
        lqx.expr_eval(psi, L(chi))                                        # psi = chi
        terms = hop_terms(psi)
        lqx.expr_eval(h, terms[0])                                        # h_smear  = ...   (E1)
        for t in terms[1:]:
            lqx.expr_eval(h, t, accumulate=True)                          # h_smear += ...   (E2)
        lqx.expr_eval(chi, L(s0) + kappa * L(h))                          # chi = s_0 + kappa*h_smear (E3)
    lqx.expr_eval(chi, (1.0 / norm) * L(chi))                             # chi /= norm (E4; reciprocal multiply, A22)


def _extras(torch, lqx, li, hbm_gbs, tune=None):
    """Per-kernel numbers for the other BASELINE configs (same JSON line, key "kernels"): device time
    per launch, algorithmic GB/s (SURVEY 8(d) bytes/site) and its fraction of the measured HBM peak.
    tune: dict that receives the lqx_autotune tables of the hop / Jacobi geometries (Figs. 1-2 on B200)."""
    out = []
    tune = {} if tune is None else tune
    flush = torch.zeros(64 * 1024 * 1024, dtype=torch.float32, device="cuda")  # 256 MB > L2

    def add(name, prec, sites, reals_per_site, flops_per_site, fn, reps=10, cold=False, lat=None, kclass=None):
        """`ms` = the whole C-ABI call (for the synchronising entry points that includes the host sync);
        with lat/kclass also `kernel_ms` = device time of that call's kernels (CUDA event pairs the
        library records around its launches)."""
        for _ in range(3):
            fn()
        torch.cuda.synchronize()
        if kclass is not None:
            lat.set_option("time_kernels", 1)
            lat.kernel_time(kclass)
        med, best = _time_kernel(torch, fn, reps, flush if cold else None)
        nbytes = sites * reals_per_site * (4 if prec == "f32" else 8)
        row = {"kernel": name, "dtype": prec, "ms": round(med, 5), "ms_best": round(best, 5),
               "site_evals_per_s": sites / (med * 1e-3), "alg_gbs": nbytes / (med * 1e-3) / 1e9,
               "hbm_frac": nbytes / (med * 1e-3) / 1e9 / hbm_gbs, "gflops": sites * flops_per_site / (med * 1e-3) / 1e9,
               "l2": "flushed between launches" if cold else "inputs larger than L2"}
        if kclass is not None:
            kms, n = lat.kernel_time(kclass)
            lat.set_option("time_kernels", 0)
            if n:
                row["kernel_ms"] = round(kms / n, 5)
                row["kernel_hbm_frac"] = nbytes / (kms / n * 1e-3) / 1e9 / hbm_gbs
        out.append(row)

    # ---- C1: 4^4 fp64, one smear step + plaquette (256 sites: launch latency, exempt from any roofline reading)
    dims = li.CONFIGS["c1"]["dims"]
    with lqx.Lattice(dims) as lat:
        u, _ = _gen_links(lat, lqx, li, "c1", "haar", "f64")
        o = [lat.alloc(lqx.COLORMAT, lqx.F64) for _ in range(4)]
        add("smear_step c1 (4^4: launch-latency-bound)", "f64", lat.volume, 144, SMEAR_CANONICAL_FLOPS, lambda: lqx.smear_step(o, u, ALPHA), reps=20)
        add("smear_step+plaquette(in) fused c1 (incl. sync)", "f64", lat.volume, 144, SMEAR_CANONICAL_FLOPS + 108,
            lambda: lqx.smear_step(o, u, ALPHA, want_plaq_in=True), reps=20)
    # ---- C2: hop, 16^3x32 fp32 (working set 63 MB < L2: cold and warm)
    dims = li.CONFIGS["c2"]["dims"]
    with lqx.Lattice(dims) as lat:
        u, _ = _gen_links(lat, lqx, li, "c2", "haar", "f32")
        psi = lat.alloc(lqx.FERMION, lqx.F32).import_dev(li.gaussian_field(2, 10, dims, "f", "f32", device="cuda"))
        chi = lat.alloc(lqx.FERMION, lqx.F32)
        v = lat.volume
        tune["hop_and_jacobi_step_16^3x32_f32"] = lat.autotune(lqx.K_HOP, lqx.F32, 5)
        # what a single L2-cold launch of this size can reach at all when timed by events: a plain copy moving the same
        # 63 MB (31.5 MB read + 31.5 MB written), measured the same way -- the event pair alone costs ~6 us
        ca = torch.empty(v * 120 // 2, dtype=torch.float32, device="cuda")
        cb = torch.empty_like(ca)
        add("copy of the same 63 MB, torch (L2-cold): the floor of one cold launch timed by events", "f32", v, 120, 0,
            lambda: cb.copy_(ca), reps=20, cold=True)
        copy_ms = out[-1]["ms"]
        del ca, cb
        add("hop c2 (L2-cold)", "f32", v, 120, 2280, lambda: lqx.hop(chi, u, psi), reps=20, cold=True)
        out[-1]["l2"] = "flushed between launches"
        out[-1]["frac_of_copy_same_bytes"] = copy_ms / out[-1]["ms"]
        add("hop c2 (L2-warm)", "f32", v, 120, 2280, lambda: lqx.hop(chi, u, psi), reps=20)
        out[-1]["l2"] = "warm: 63 MB working set fits the 126 MB L2"
        def hop20():
            for _ in range(20):
                lqx.hop(chi, u, psi)

        add("hop c2, 20 launches back to back (per 20; ramp-up and drain overlap as in the iterated Jacobi routine)", "f32", v * 20, 120, 2280,
            hop20, reps=10)
        out[-1]["l2"] = "warm: 63 MB working set fits the 126 MB L2"
        # "CUDA-graph-amortised" -- the same 20 launches captured once and replayed as one graph
        try:
            side = torch.cuda.Stream()
            lat.set_stream(side)
            with torch.cuda.stream(side):
                lqx.hop(chi, u, psi)
                side.synchronize()
                graph = torch.cuda.CUDAGraph()
                with torch.cuda.graph(graph, stream=side):
                    hop20()
                add("hop c2, 20 launches replayed as ONE CUDA graph (per 20)", "f32", v * 20, 120, 2280, graph.replay, reps=10)
                out[-1]["l2"] = "warm: 63 MB working set fits the 126 MB L2"
                del graph
        except Exception as e:  # a failed capture must not take the bench line down
            out.append({"kernel": "hop c2, CUDA graph", "error": repr(e)[:200]})
        finally:
            torch.cuda.synchronize()
            lat.set_stream(torch.cuda.current_stream())
        add("hop+norm2 fused c2 (L2-cold, incl. sync)", "f32", v, 120, 2328, lambda: lqx.hop_norm2(chi, u, psi), reps=20, cold=True,
            lat=lat, kclass=lqx.K_HOP)
    # ---- the same hop kernel on a lattice 16x larger (32^3x64: 1 GB moved), where launch ramp-up and
    # drain no longer dominate: the kernel's own HBM fraction
    dims = li.CONFIGS["c5"]["dims"]
    for prec, pcode in (("f32", lqx.F32), ("f64", lqx.F64)):
        with lqx.Lattice(dims) as lat:
            u = []
            for mu in range(4):
                a = li._as_real(li.haar_su3_complex(2, mu, lat.volume, "cuda"), prec)
                u.append(lat.alloc(lqx.COLORMAT, pcode).import_dev(a))
                del a
            psi = lat.alloc(lqx.FERMION, pcode).import_dev(li.gaussian_field(2, 10, dims, "f", prec, device="cuda"))
            chi = lat.alloc(lqx.FERMION, pcode)
            tune[f"hop_and_jacobi_step_32^3x64_{prec} (the lattice of the paper's Figs. 1-2)"] = lat.autotune(lqx.K_HOP, pcode, 3)
            add("hop 32^3x64 (not a BASELINE config; size check)", prec, lat.volume, 120, 2280, lambda: lqx.hop(chi, u, psi), reps=10)
            eh = None
            for mu in range(4):  # the Listing's E1/E2 expression, summed over mu, as ONE run-time expression
                t = lqx.Expr.leaf(u[mu]) * lqx.shifted(psi, lqx.FORWARD, mu) + lqx.shifted(lqx.adj(u[mu]) * lqx.Expr.leaf(psi), lqx.BACKWARD, mu)
                eh = t if eh is None else eh + t
            lqx.expr_eval(chi, eh)
            add("hop 32^3x64 as a run-time expression (NVRTC)", prec, lat.volume, 120, 2280, lambda: lqx.expr_eval(chi, eh), reps=10)
    # ---- NEXT-1: the paper's complete Jacobi smearing routine at its Table 1 sizes 16^3x32 and 32^3x64
    # (PAPER.md:228-238), fermion field, 20 iterations, all four directions.  Per iteration and site the fused
    # kernel moves U 72 + psi 24 + s_0 24 + chi 24 = 144 reals and does 2280 (hop) + 48 (E3) canonical flops.
    JIT = 20
    for dims in (li.CONFIGS["c2"]["dims"], li.CONFIGS["c5"]["dims"]):
        for prec, pcode in (("f32", lqx.F32), ("f64", lqx.F64)):
            with lqx.Lattice(dims) as lat:
                u = []
                for mu in range(4):
                    a = li._as_real(li.haar_su3_complex(2, mu, lat.volume, "cuda"), prec)
                    u.append(lat.alloc(lqx.COLORMAT, pcode).import_dev(a))
                    del a
                chi = lat.alloc(lqx.FERMION, pcode).import_dev(li.gaussian_field(2, 10, dims, "f", prec, device="cuda"))
                tmp = [lat.alloc(lqx.FERMION, pcode) for _ in range(2)]
                add(f"jacobi_smear {dims[0]}^3x{dims[3]} x{JIT} iterations (NEXT-1; paper Table 1 size)", prec, lat.volume * JIT,
                    144, 2328, lambda: lqx.jacobi_smear(chi, u, 0.01, JIT, -1, 1.0, tmp), reps=10)
                out[-1]["l2"] = "iterated on resident fields (working set %.0f MB)" % (lat.volume * 168 * (4 if prec == "f32" else 8) / 1e6)
                out[-1]["paper_gflops_gtx480"] = {(16, "f32"): 11.86, (16, "f64"): 6.26, (32, "f32"): 21.31}.get((dims[0], prec))
                if dims[0] == 32:  # the same routine as user code on the run-time expression path (NEXT-2)
                    work = [lat.alloc(lqx.FERMION, pcode) for _ in range(3)]
                    for fused, label in ((True, "one run-time expression per iteration"), (False, "Listing 1 literally: E0..E4 as six run-time expressions per iteration")):
                        jacobi_listing(lqx, chi, u, 0.01, 1, -1, 1.0, work, fused)  # compiles the kernels
                        add(f"jacobi_smear {dims[0]}^3x{dims[3]} x{JIT} iterations, {label}", prec, lat.volume * JIT, 144, 2328,
                            lambda: jacobi_listing(lqx, chi, u, 0.01, JIT, -1, 1.0, work, fused), reps=5)
                        out[-1]["l2"] = "fused: 144 reals per site and iteration; literal listing: 24+24 (E0) + 66+3*90 (E1,E2) + 72 (E3) = 456"
    # ---- C3: smear + plaquette, 32^3x64 fp64
    dims = li.CONFIGS["c3"]["dims"]
    with lqx.Lattice(dims) as lat:
        u, _ = _gen_links(lat, lqx, li, "c3", "haar", "f64")
        o = [lat.alloc(lqx.COLORMAT, lqx.F64) for _ in range(4)]
        v = lat.volume
        add("smear_step c3", "f64", v, 144, SMEAR_CANONICAL_FLOPS, lambda: lqx.smear_step(o, u, ALPHA), reps=12)
        add("smear_step+plaquette(in) fused c3 (incl. sync)", "f64", v, 144, SMEAR_CANONICAL_FLOPS + 108,
            lambda: lqx.smear_step(o, u, ALPHA, want_plaq_in=True), reps=12, lat=lat, kclass=lqx.K_SMEAR)
        add("plaquette c3 (incl. sync)", "f64", v, 72, 2591, lambda: lqx.plaquette(u), reps=6, lat=lat, kclass=lqx.K_PLAQUETTE)
        # the same quantity stated by the user as an expression and reduced inside ONE generated kernel
        L = lqx.Expr.leaf
        pe = None
        for mu in range(3):
            for nu in range(mu + 1, 4):
                t = (L(u[mu]) * lqx.shifted(u[nu], lqx.FORWARD, mu)) * lqx.adj(L(u[nu]) * lqx.shifted(u[mu], lqx.FORWARD, nu))
                pe = t if pe is None else pe + t
        pe = pe.trace()
        lqx.expr_reduce(lqx.R_SUM, pe)  # compiles
        add("plaquette c3 as a run-time expression: sum(trace(sum_{mu<nu} ...)) in one generated kernel (incl. sync)", "f64", v, 72, 2591,
            lambda: lqx.expr_reduce(lqx.R_SUM, pe), reps=6, lat=lat, kclass=lqx.K_REDUCE)
    # ---- C5: catalogue sweep, 32^3x64, both precisions
    dims = li.CONFIGS["c5"]["dims"]
    for prec, pcode in (("f32", lqx.F32), ("f64", lqx.F64)):
        with lqx.Lattice(dims) as lat:
            v = lat.volume
            cm = [lat.alloc(lqx.COLORMAT, pcode).import_dev(li.gaussian_field(7, k, dims, "cm", prec, device="cuda")) for k in range(4)]
            vec = lat.alloc(lqx.COLORVEC, pcode).import_dev(li.gaussian_field(7, 4, dims, "cv", prec, device="cuda"))
            r = lat.alloc(lqx.COLORMAT, pcode)
            c = lat.alloc(lqx.COMPLEX, pcode)
            w = lat.alloc(lqx.COLORVEC, pcode)
            torch.cuda.synchronize()
            add("form i  A*B+C*adj(D) c5", prec, v, 90, 414, lambda: lqx.mm_plus_madj(r, cm[0], cm[1], cm[2], cm[3]))
            add("form ii trace(A*B) c5", prec, v, 38, 70, lambda: lqx.trace_mm(c, cm[0], cm[1]))
            add("form iii 2.5*A-shift(B,BACKWARD,2) c5", prec, v, 54, 36, lambda: lqx.ax_minus_shift(r, 2.5, cm[0], cm[1], lqx.BACKWARD, 2))
            add("form iii' 2.5*A-shift(B,FORWARD,0) c5", prec, v, 54, 36, lambda: lqx.ax_minus_shift(r, 2.5, cm[0], cm[1], lqx.FORWARD, 0))
            add("form iv M*v c5", prec, v, 30, 66, lambda: lqx.mat_vec(w, cm[0], vec))
            # NEXT-2: the same forms as run-time expressions (one NVRTC-compiled fused kernel each, cached)
            e1 = lqx.Expr.leaf(cm[0]) * lqx.Expr.leaf(cm[1]) + lqx.Expr.leaf(cm[2]) * lqx.adj(cm[3])
            t0 = time.perf_counter()
            lqx.expr_eval(r, e1)
            torch.cuda.synchronize()
            jit_s = time.perf_counter() - t0
            add("form i  as a run-time expression (NVRTC) c5", prec, v, 90, 414, lambda: lqx.expr_eval(r, e1))
            out[-1]["first_use_compile_s"] = round(jit_s, 3)
            add("norm2(A*B+C*adj(D)) fused into one generated kernel (incl. sync)", prec, v, 72, 414 + 36,
                lambda: lqx.expr_reduce(lqx.R_NORM2, e1), lat=lat, kclass=lqx.K_REDUCE)
            add("sum(trace(A*B)) fused into one generated kernel (incl. sync)", prec, v, 36, 70 + 2,
                lambda: lqx.expr_reduce(lqx.R_SUM, (lqx.Expr.leaf(cm[0]) * lqx.Expr.leaf(cm[1])).trace()), lat=lat, kclass=lqx.K_REDUCE)
            e3 = 2.5 * lqx.Expr.leaf(cm[0]) - lqx.shifted(cm[1], lqx.BACKWARD, 2)
            add("form iii as a run-time expression (NVRTC) c5", prec, v, 54, 36, lambda: lqx.expr_eval(r, e3))
            add("shift(A,FORWARD,3) c5", prec, v, 36, 0, lambda: lqx.shift(r, cm[0], lqx.FORWARD, 3))
            add("norm2(colour matrix) c5 (incl. sync)", prec, v, 18, 36, lambda: lqx.norm2(cm[0]), lat=lat, kclass=lqx.K_REDUCE)
            add("sum(colour matrix) c5 (incl. sync)", prec, v, 18, 18, lambda: lqx.sum(cm[0]), lat=lat, kclass=lqx.K_REDUCE)
            add("trace(colour matrix) c5 (incl. sync)", prec, v, 6, 6, lambda: lqx.trace(cm[0]), lat=lat, kclass=lqx.K_REDUCE)
    del flush
    torch.cuda.empty_cache()
    return out


def run_sweep(args):
    """NEXT-3: the paper's launch-geometry experiment (Figs. 1 and 2: performance against
    N_threads for N_site in {1,2,4,8} and against N_site for N_threads in {32,..,256}, on E2 at 32^3x64 SP) redone
    on the fused Jacobi iteration: P(N_threads, N_site) in GFLOPS (canonical 2328 flops per site and iteration)
    and as a fraction of the HBM roofline.  Prints one JSON line with key "geometry_sweep"."""
    import torch

    import lattice_inputs as li
    import paper_1105_2279_b200 as lqx

    hbm_gbs = _peaks()[0]
    dims = li.CONFIGS["c5"]["dims"]  # 32^3x64, the paper's sweep lattice
    rows = []
    iters = 20
    for prec, pcode in (("f32", lqx.F32), ("f64", lqx.F64)):
        with lqx.Lattice(dims) as lat:
            u = []
            for mu in range(4):
                a = li._as_real(li.haar_su3_complex(2, mu, lat.volume, "cuda"), prec)
                u.append(lat.alloc(lqx.COLORMAT, pcode).import_dev(a))
                del a
            chi = lat.alloc(lqx.FERMION, pcode).import_dev(li.gaussian_field(2, 10, dims, "f", prec, device="cuda"))
            tmp = [lat.alloc(lqx.FERMION, pcode) for _ in range(2)]
            for nthreads in (32, 64, 128, 256):
                for nsite in (1, 2, 4):
                    lat.set_option("jacobi_block", nthreads)
                    lat.set_option("jacobi_sites", nsite)
                    fn = lambda: lqx.jacobi_smear(chi, u, 0.01, iters, -1, 1.0, tmp)
                    for _ in range(3):
                        fn()
                    torch.cuda.synchronize()
                    med, best = _time_kernel(torch, fn, 7)
                    per_it = med / iters
                    nbytes = lat.volume * 144 * (4 if prec == "f32" else 8)
                    rows.append({"dtype": prec, "n_threads": nthreads, "n_site": nsite, "us_per_iteration": round(per_it * 1e3, 2),
                                 "gflops": lat.volume * 2328 / (per_it * 1e-3) / 1e9, "hbm_frac": nbytes / (per_it * 1e-3) / 1e9 / hbm_gbs})
    best = {p: max((r for r in rows if r["dtype"] == p), key=lambda r: r["gflops"]) for p in ("f32", "f64")}
    print(json.dumps({"geometry_sweep": {"kernel": "k_jacobi_step (one fused Jacobi iteration, fermion)", "dims": list(dims), "rows": rows,
                                         "best": best, "paper": "GTX 480: N_threads = 32 best for every expression, N_site 4 or 8 "
                                                                "slightly better than 1 (PAPER.md:248, :260)"}}))


def _kernel_only_other(args, torch, lqx, li, lat, u):
    """--kernel-only --only plaquette|hop|reduce: a few launches of that kernel on the workload's lattice (what ncu wraps)."""
    P = u[0].prec
    if args.only == "reduce":
        # the three standalone reductions on one link field of the workload's lattice, kernel time from the library's own
        # event pairs (--workload c3: the 32^3x64 fp64 colour matrix of the configs[4] rows)
        lat.set_option("time_kernels", 1)
        rows = {}
        for name, call in (("norm2", lqx.norm2), ("sum", lqx.sum), ("trace", lqx.trace)):
            for _ in range(3):
                call(u[0])
            lat.kernel_time(lqx.K_REDUCE)
            for _ in range(max(args.steps, 3)):
                call(u[1]), call(u[2]), call(u[3]), call(u[0])  # four fields in turn
            ms, n = lat.kernel_time(lqx.K_REDUCE)
            rows[name] = ms / n
        print(json.dumps({"kernel_only": "reduce", "workload": args.workload, "kernel_ms": rows}))
        lat.close()
        return
    if args.only == "plaquette":
        fn = lambda: lqx.plaquette(u)
    else:
        psi = lat.alloc(lqx.FERMION, P).import_dev(li.gaussian_field(2, 10, lat.dims, "f", "f32" if P == lqx.F32 else "f64", device="cuda"))
        chi = lat.alloc(lqx.FERMION, P)
        fn = lambda: lqx.hop(chi, u, psi)
    for _ in range(3):
        fn()
    torch.cuda.synchronize()
    med, best = _time_kernel(torch, fn, max(args.steps, 3))
    print(json.dumps({"kernel_only": args.only, "workload": args.workload, "ms": med, "ms_best": best}))
    lat.close()


def run_tsplit(args):
    """NEXT-4: ONE global lattice decomposed along t over the ranks, halo exchange over
    torch.distributed (NCCL) overlapped with the interior launch (paper_1105_2279_b200/tsplit.py).  Not the contract
    (BASELINE.json: replicas only) -- an extra mode: `torchrun ... bench.py --tsplit --gpus N`; with one GPU the halos
    are the rank's own periodic images, which measures what the split formulation costs by itself."""
    import torch

    import lattice_inputs as li
    import paper_1105_2279_b200 as lqx
    from paper_1105_2279_b200 import tsplit

    rank, world, local, barrier, vmax = _dist()
    torch.cuda.set_device(local)
    wl = WORKLOADS[args.workload]
    cfg = li.CONFIGS[wl["cfg"]]
    gdims, prec = cfg["dims"], cfg["prec"]
    P = lqx.F32 if prec == "f32" else lqx.F64
    K, W = args.steps, max(args.warmup, 3)
    ldims = tsplit.local_dims(gdims, world)
    lat = lqx.Lattice(ldims, device=local)
    comm = tsplit.DistComm() if world > 1 else tsplit.SelfComm()
    ts = tsplit.TSplit(tsplit.LqxBackend(lqx, lat), comm, gdims)
    # synthetic links of the workload's recipe on the local lattice (own slices and halos alike; the first exchange
    # overwrites the halos): timing does not depend on which slab of the global field a rank holds
    u = []
    for mu in range(4):
        z = (li.near_unit_su3_complex(cfg["seed"] + 100 * rank, mu, lat.volume, 0.1, f"cuda:{local}") if wl["recipe"] == "near_unit"
             else li.haar_su3_complex(cfg["seed"] + 100 * rank, mu, lat.volume, f"cuda:{local}"))
        a = li._as_real(z, prec)
        u.append(lat.alloc(lqx.COLORMAT, P).import_dev(a))
        del z, a
    tmp = [lat.alloc(lqx.COLORMAT, P) for _ in range(4)]
    torch.cuda.synchronize()
    for _ in range(W):
        ts.smear_step(tmp, u, ALPHA)
        u, tmp = tmp, u
    torch.cuda.synchronize()
    barrier()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record()
    for _ in range(K):
        ts.smear_step(tmp, u, ALPHA)
        u, tmp = tmp, u
    e1.record()
    torch.cuda.synchronize()
    barrier()
    ms = vmax(e0.elapsed_time(e1))
    plaq = ts.plaquette_sum(u) / (18.0 * li.volume(gdims))
    V = li.volume(gdims)
    esize = 4 if prec == "f32" else 8
    if rank == 0:
        print(json.dumps({
            "metric": "smear-step site-updates/s", "value": V * K / (ms * 1e-3), "unit": "site-updates/s", "n_gpus": world,
            "steps": K, "warmup": W, "ms_per_step": ms / K, "higher_is_better": True, "scaling": "strong", "vs_baseline": None,
            "dtype": prec, "data": "synthetic", "mode": "tsplit",
            "config": {"workload": wl["desc"] + " -- ONE lattice decomposed along t", "dims": list(gdims), "local_dims": list(ldims),
                       "parallelism": f"t-split x{world}: per step and rank 2 x 4 halo slices = "
                                      f"{2 * 4 * ldims[0] * ldims[1] * ldims[2] * 18 * esize / 1e6:.1f} MB exchanged "
                                      + ("over NCCL" if world > 1 else "(one rank: its own periodic images, device copies)")
                                      + ", overlapped with the interior launch", "l2": "inputs larger than L2"},
            "plaquette_avg_after_last_step": plaq}))
    lat.close()
    if world > 1:
        import torch.distributed as dist

        dist.destroy_process_group()


def run_ours(args):
    import torch

    import lattice_inputs as li
    import paper_1105_2279_b200 as lqx

    rank, world, local, barrier, vmax = _dist()
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: the lqx library has no CPU fallback")
    torch.cuda.set_device(local)
    wl = WORKLOADS[args.workload]
    cfg = li.CONFIGS[wl["cfg"]]
    dims, prec = cfg["dims"], cfg["prec"]
    esize = 4 if prec == "f32" else 8
    K, W = args.steps, max(args.warmup, 3)
    hbm_gbs, hbm_src, sm_max = _peaks()
    want_host = not args.kernel_only  # e2e (every rank) and cpu_baseline (rank 0 at N = 1) need the host copy

    lat = lqx.Lattice(dims, device=local)
    V = lat.volume
    u, host = _gen_links(lat, lqx, li, wl["cfg"], wl["recipe"], prec, keep_host=want_host)
    tmp = [lat.alloc(lqx.COLORMAT, u[0].prec) for _ in range(4)]

    # roofline denominators measured in this run (reported beside the driver-written peak)
    fma_kind = 0 if prec == "f32" else 2
    fma_peak = lat.bench_fma_peak(fma_kind)
    fma2_peak = lat.bench_fma_peak(1) if prec == "f32" else None
    copy_peak = lat.bench_copy_peak(1 << 30)
    # the FMA pipe fed the way the kernel feeds it: 3x3 complex products on register operands (three distinct register
    # operands per instruction, FFMA2 with broadcast / swapped operands in fp32) instead of one dependent chain
    prod_peak = lat.bench_fma_peak(3 if prec == "f32" else 4)

    if args.smear_variant:
        lat.set_option("smear_variant", args.smear_variant)
    if args.tile >= 0:
        lat.set_option("tile", args.tile)
    for kv in args.opt:  # any other library option, e.g. --opt bulk_fill=1 (reproducible captures of optional code paths)
        k, v = kv.split("=")
        lat.set_option(k, int(v))
    if args.block:
        lat.set_option("block", args.block)
    tune_tables = None
    if args.autotune or (world == 1 and not args.kernel_only and not args.smear_variant):
        # NEXT-3: the library times its launch geometries on this lattice and keeps the winners;
        # the tables go into the JSON line (the B200 counterpart of the paper's Figs. 1-2)
        tune_tables = {"smear": lat.autotune(lqx.K_SMEAR, u[0].prec, 3), "plaquette": lat.autotune(lqx.K_PLAQUETTE, u[0].prec, 3)}
    if args.kernel_only and args.only != "smear":
        return _kernel_only_other(args, torch, lqx, li, lat, u)

    lqx.smear_iterate(u, tmp, ALPHA, W)  # warm-up (>= 3 steps)
    torch.cuda.synchronize()
    lat.set_option("time_kernels", 1)
    lat.kernel_time(lqx.K_SMEAR), lat.kernel_time(lqx.K_PLAQUETTE)
    sampler = ClockSampler(local)
    barrier()
    torch.cuda.synchronize()
    launches0 = lat.launch_count()
    sampler.start()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record()
    plaqs = lqx.smear_iterate(u, tmp, ALPHA, K)  # K steps, plaquette after each; syncs once at the end
    e1.record()
    torch.cuda.synchronize()
    barrier()
    clocks = sampler.stop()
    ms = vmax(e0.elapsed_time(e1))
    launches = lat.launch_count() - launches0
    smear_ms, smear_n = lat.kernel_time(lqx.K_SMEAR)
    plaq_ms, plaq_n = lat.kernel_time(lqx.K_PLAQUETTE)
    lat.set_option("time_kernels", 0)

    value = replica_value(world, V, K, ms)
    k_ms = smear_ms / max(smear_n, 1)  # average duration of the dominant kernel inside the timed region
    alg_bytes = V * SMEAR_REALS_PER_SITE * esize
    # the kernel that actually ran (options, tuned choice and fall-backs resolved by the library) and what it executes
    variant, lane_ops_site, kname = lat.smear_info()
    lane_ops = V * lane_ops_site
    # FP-pipe peak from unit counts and clocks: 148 SMs x 128 fp32 (64 fp64) FMA lanes x sm_max
    alu_peak_tflops = 148 * (128 if prec == "f32" else 64) * 2 * sm_max * 1e6 / 1e12
    cap, cap_src = _ncu_capture(kname, prec)
    traffic = (cap["dram__bytes_read.sum"] + cap["dram__bytes_write.sum"]) if cap else None
    # `achieved` counts the ALGORITHMIC work of a site update -- SURVEY.md 8(d): the literal evaluation's 48 products + update =
    # 5328 FMA lane-ops per site -- whatever order the kernel evaluates it in (a kernel that needs fewer products for the
    # same update is faster against the same ceiling); the lane-ops the kernel actually EXECUTES (lqx_smear_info; 4680 for
    # the 42-product orders) are reported beside it as the utilisation of the FMA pipe
    alg_lane_ops = V * SMEAR_LANE_OPS_LITERAL
    alu_frac = 2 * alg_lane_ops / (k_ms * 1e-3) / 1e12 / alu_peak_tflops
    exe_frac = 2 * lane_ops / (k_ms * 1e-3) / 1e12 / alu_peak_tflops
    hbm_frac = alg_bytes / (k_ms * 1e-3) / 1e9 / hbm_gbs
    roofline = {
        "kernel": f"{kname} (staple sum + smear update of all four links, fused input plaquette; smear_variant {variant})",
        "bound": "alu", "achieved": 2 * alg_lane_ops / (k_ms * 1e-3) / 1e12, "peak": alu_peak_tflops, "unit": "TFLOP/s",
        "frac": alu_frac,
        "executed": {"lane_ops_per_site": lane_ops_site, "achieved": 2 * lane_ops / (k_ms * 1e-3) / 1e12, "frac": exe_frac,
                     "what": "FMA lane-ops the kernel that ran executes (lqx_smear_info) x 2 / kernel time: the FMA pipe's utilisation"},
        "peak_source": f"148 SMs x {128 if prec == 'f32' else 64} FMA lanes x 2 x {sm_max:.0f} MHz (DESIGN.md sec.7); "
                       f"FMA-chain micro-benchmark in this run: {2 * fma_peak / 1e12:.1f} TFLOP/s"
                       + (f", packed f32x2: {2 * fma2_peak / 1e12:.1f}" if fma2_peak else ""),
        "frac_at_measured_clock": alu_frac / (clocks["sm_mhz"] / sm_max) if clocks.get("sm_mhz") else None,
        "product_stream_peak_tflops": 2 * prod_peak / 1e12,
        "frac_of_product_stream_peak": (2 * lane_ops / (k_ms * 1e-3)) / (2 * prod_peak),
        "flops_counted": f"algorithmic: {SMEAR_LANE_OPS_LITERAL} FMA lane-ops x 2 per site update (SURVEY.md 8(d), literal 48-product evaluation); "
                         f"this kernel executes {lane_ops_site} (see `executed`; frac_of_product_stream_peak uses the executed count)",
        "traffic": traffic, "traffic_unit": "bytes per launch (ncu dram__bytes_read.sum + dram__bytes_write.sum)",
        "traffic_source": cap_src, "ms_per_launch": k_ms, "launches": smear_n,
        "hbm": {"bound": "hbm", "achieved": alg_bytes / (k_ms * 1e-3) / 1e9, "peak": hbm_gbs, "unit": "GB/s",
                "frac": hbm_frac, "peak_source": hbm_src,
                "copy_kernel_this_run_gbs": copy_peak / 1e9, "alg_bytes_per_launch": alg_bytes},
        # neither roof is what the kernel runs into: ncu names the unit; from the committed capture
        "busiest_units_ncu": ({k: cap[k] for k in ("l1tex__data_pipe_lsu_wavefronts.avg.pct_of_peak_sustained_elapsed",
                                                   "smsp__issue_active.avg.pct_of_peak_sustained_active",
                                                   "sm__pipe_fma_cycles_active.avg.pct_of_peak_sustained_active",
                                                   "lts__throughput.avg.pct_of_peak_sustained_elapsed",
                                                   "gpu__dram_throughput.avg.pct_of_peak_sustained_elapsed") if k in cap}
                              if cap else None),
        "l1_data_pipe_ceiling": "128 B/clk/SM = 32 fp32 operands per clock for 128 FMA lanes: the literal evaluation moves "
                                "76 matrices x 72 B per site through it (42.8 clk/site) for 5328 lane-ops (41.6 clk/site)",
        "north_star_target": {"text": "smear step >= 70 % of the HBM roofline", "hbm_frac": hbm_frac, "met": bool(hbm_frac >= 0.70)},
    }
    line = {
        "metric": "smear-step site-updates/s", "value": value, "unit": "site-updates/s", "n_gpus": world,
        "steps": K, "warmup": W, "ms_per_step": ms / K, "higher_is_better": True, "scaling": "weak",
        "vs_baseline": None, "dtype": prec, "data": "synthetic",
        "config": {"workload": wl["desc"], "dims": list(dims), "sites": V, "alpha": ALPHA, "l2": "inputs larger than L2 "
                   f"({2 * alg_bytes / 2 / 1e9:.2f} GB read+written per step)", "parallelism": "replicas only" if world > 1 else "1 GPU",
                   "smear_variant": variant, "smear_kernel": kname},
        "gflops_canonical": world * V * K * SMEAR_CANONICAL_FLOPS / (ms * 1e-3) / 1e9,
        "hbm_gbs_algorithmic": world * (K * alg_bytes + V * PLAQ_REALS_PER_SITE * esize) / (ms * 1e-3) / 1e9,
        "plaquette_avg_after_each_step": plaqs,
        "clocks": clocks, "gpu_launches": launches, "roofline": roofline,
        "step_breakdown_ms": {"smear_kernels": smear_ms, "plaquette_kernel": plaq_ms, "smear_launches": smear_n,
                              "plaquette_launches": plaq_n, "timed_region": ms},
    }

    if tune_tables is not None:
        line["autotune"] = {"what": "lqx_autotune on this lattice: ms per launch of every candidate geometry, chosen = kept "
                                    "(param: smear = [smear_variant, tile], plaquette = [plaq_variant, 0])", **tune_tables}
    if not args.kernel_only:
        # ---- e2e: the public host-buffer call, H2D + D2H inside the timed region, every step; under torchrun every
        # rank runs its replica from its own pinned buffers and the job takes as long as the slowest rank
        hin = host
        hout = [torch.empty(h.shape, dtype=h.dtype, pin_memory=True) for h in host]
        lqx.smear_iterate_host(lat, u[0].prec, hin, hout, ALPHA, 1)  # warm-up
        torch.cuda.synchronize()
        ke = min(K, args.e2e_steps)
        barrier()
        t0 = time.perf_counter()
        for _ in range(ke):
            lqx.smear_iterate_host(lat, u[0].prec, hin, hout, ALPHA, 1)
            hin, hout = hout, hin
        torch.cuda.synchronize()
        te = vmax(time.perf_counter() - t0)
        barrier()
        fbytes = V * 18 * esize * 4
        line["e2e"] = {"value": replica_value(world, V, ke, te * 1e3), "unit": "site-updates/s", "h2d_bytes_per_step": world * fbytes,
                       "d2h_bytes_per_step": world * (fbytes + 8), "steps": ke, "ms_per_step": te / ke * 1e3,
                       "call": "lqx_smear_iterate_host(nsteps=1) on pinned host buffers in QDP order (time-slice slabs streamed: upload / step / download overlap)"}
        del hout, hin
    else:
        line["e2e"] = None
    if world == 1 and not args.kernel_only:
        # ---- cpu baseline: the oracle on this box's host cores
        import oracle as orc

        line["cpu_baseline"] = _cpu_baseline(orc, dims, prec, host)
    for f in u + tmp:
        f.free()
    lat.close()
    torch.cuda.empty_cache()
    if world == 1 and not args.no_extras and not args.kernel_only:
        more = {}
        line["kernels"] = _extras(torch, lqx, li, hbm_gbs, more)
        line.setdefault("autotune", {"what": "lqx_autotune"}).update(more)
        line["autotune"]["what_hop"] = ("hop tables: param[0] > 0 = CTA size of lqx_hop; param[0] < 0 = N_threads = -param[0], "
                                        "N_site = param[1] of one lqx_jacobi_smear iteration (PAPER.md:117-126), ms per iteration")
    if rank == 0:
        print(json.dumps(line))
    if world > 1:
        import torch.distributed as dist

        dist.destroy_process_group()


def run_reference(args):
    """The oracle, as it stands, on this box's host cores: each step = one bounded sample of the workload
    (smear update of all four links + plaquette integrand on the first n sites of the full-size field)."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    import numpy as np

    import lattice_inputs as li
    import oracle as orc

    wl = WORKLOADS[args.workload]
    cfg = li.CONFIGS[wl["cfg"]]
    dims, prec = cfg["dims"], cfg["prec"]
    V = li.volume(dims)
    # the sample only touches sites within one time-slice of its range, but the oracle indexes the full
    # lattice: generate the whole field (on the GPU if there is one -- input generation only)
    try:
        import torch

        dev = "cuda" if torch.cuda.is_available() else "cpu"
    except Exception:
        dev = "cpu"
    u = [t.cpu().numpy() for t in li.gauge_field(cfg["seed"], dims, prec, wl["recipe"], device=dev)]
    variant = orc.native_variant(prec)
    n = min(V, args.ref_sites)
    sites = np.repeat(np.arange(n, dtype=np.int64), 4)
    mus = np.tile(np.arange(4, dtype=np.int32), n)
    only = np.arange(n, dtype=np.int64)

    def step():
        orc.smear_links(dims, u, ALPHA, sites, mus, variant)
        orc.plaquette_sites(dims, u, only, variant)

    K, W = args.steps, args.warmup
    for _ in range(W):
        step()
    t0 = time.perf_counter()
    for _ in range(K):
        step()
    t = time.perf_counter() - t0
    value = n * K / t
    sample = f"each step: first {n} of {V} sites (all 4 directions + plaquette), oracle variant {variant}"
    print(json.dumps({
        "impl": "reference", "metric": "smear-step site-updates/s", "value": value, "unit": "site-updates/s",
        "n_gpus": int(os.environ.get("WORLD_SIZE", "1")), "steps": K, "warmup": W, "ms_per_step": t / K * 1e3,
        "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": prec, "data": "synthetic",
        "config": {"workload": wl["desc"], "dims": list(dims), "sites": V, "alpha": ALPHA},
        "cpu_baseline": {"value": value, "unit": "site-updates/s", "cores": orc.num_threads(), "kind": "oracle", "sample": sample},
        "e2e": {"value": value, "unit": "site-updates/s", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }))


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=10)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--workload", default="c4", choices=sorted(WORKLOADS))
    ap.add_argument("--no-extras", action="store_true", help="skip the per-kernel numbers of the other configs")
    ap.add_argument("--sweep-geometry", action="store_true",
                    help="NEXT-3: P(N_threads, N_site) of the fused Jacobi iteration at 32^3x64 (the paper's Figs. 1-2)")
    ap.add_argument("--extras-only", action="store_true",
                    help="only the per-kernel numbers of configs 2, 3, 5 and the Jacobi routine (one JSON line with key "
                         "'kernels'): the command ncu wraps for the catalogue / hop / Jacobi kernels")
    ap.add_argument("--smear-variant", type=int, default=0, help="lqx option smear_variant (0 = library default / tuned)")
    ap.add_argument("--tile", type=int, default=-1, help="lqx option tile (-1 = automatic)")
    ap.add_argument("--opt", action="append", default=[], metavar="KEY=INT", help="any other lqx_set_option, repeatable")
    ap.add_argument("--block", type=int, default=0, help="lqx option block (slab thickness of the row-tile kernels)")
    ap.add_argument("--only", default="smear", choices=["smear", "plaquette", "hop", "reduce"],
                    help="with --kernel-only: the kernel to run (the command ncu wraps for that kernel)")
    ap.add_argument("--tsplit", action="store_true",
                    help="NEXT-4 extra mode: one global lattice decomposed along t over the ranks (halo exchange), not replicas")
    ap.add_argument("--autotune", action="store_true", help="let lqx_autotune pick the launch geometries before timing")
    ap.add_argument("--kernel-only", action="store_true",
                    help="timed device region only (no e2e, no cpu_baseline, no extras): the command ncu wraps")
    ap.add_argument("--e2e-steps", type=int, default=5, help="cap on host-buffer steps timed for e2e")
    ap.add_argument("--ref-sites", type=int, default=400000, help="sites per step of the --impl reference sample")
    args = ap.parse_args()
    if args.sweep_geometry:
        run_sweep(args)
    elif args.extras_only:
        import torch

        import lattice_inputs as li
        import paper_1105_2279_b200 as lqx

        print(json.dumps({"kernels": _extras(torch, lqx, li, _peaks()[0])}))
    elif args.impl == "reference":
        run_reference(args)
    elif args.tsplit:
        run_tsplit(args)
    else:
        run_ours(args)


if __name__ == "__main__":
    main()
