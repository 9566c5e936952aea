"""bench.py -- Wilson-clover Dslash throughput on B200 (BASELINE.json `metric`).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference] [--quick]

Workload: the 32^3 x 64 fp32 lattice that north_star's 70 %
bar names (BASELINE.json configs[3]'s lattice and inner precision): links by the configs[0]
recipe with eps = 0.5, stored with 12 reals, kappa = 0.1355, csw = 1.0, antiperiodic t.
A STEP is one application of the even-odd preconditioned Wilson-clover operator
    Mhat_ee = A_ee - kappa^2 H_eo A_oo^-1 H_oe
= two launches of the hopping-term kernel with the clover-inverse apply, the clover apply
and the xpay fused in their epilogues.  The headline value is the
nominal Dslash GFLOP/s (1320 flop/site per hop + 504 per clover apply; BASELINE.json
north_star) with inputs resident in HBM; `e2e` is the same operator through
qcd_dslash_host with HOST buffers.  Further objects in the same JSON line report every
other kernel of the path (plain hop 12/18-real, fp64, the fused BLAS-1 kernels) against
the HBM roofline, and CG / mixed-CG / Chebyshev timings.

Multi-GPU: the path does not shard in this build (north_star: "Everything runs on one
GPU"): `--gpus N` runs N independent replicas, one per rank, no data-path collective
(launched by torchrun, or by bench.py itself when no launcher set WORLD_SIZE).
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

DIMS = (32, 32, 32, 64)
SMALL_DIMS = (16, 16, 16, 32)          # configs[1] lattice: the oracle's bounded sample
EPS, KAPPA, CSW = 0.5, 0.1355, 1.0
HOP_FLOP, CLOVER_FLOP = 1320.0, 504.0  # nominal flop / site (north_star)
METRIC, UNIT = "wilson_clover_dslash_gflops", "GFLOP/s"
TABLE_SCALE = 1.0


def parse_args():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=1000)
    ap.add_argument("--warmup", type=int, default=20)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--quick", action="store_true", help="skip the per-kernel / solver sections")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-solvers", action="store_true", help="kernel table only (for ncu passes)")
    ap.add_argument("--solvers-only", action="store_true", help="headline step + solver table only (for ncu passes)")
    ap.add_argument("--config4", action="store_true", help="(default now) run the 48^3x96 Chebyshev workload (configs[4])")
    ap.add_argument("--no-config4", action="store_true", help="skip the 48^3x96 Chebyshev workload (configs[4])")
    ap.add_argument("--config4-only", action="store_true", help="only the configs[4] section (for ncu passes)")
    ap.add_argument("--cheb-degree", type=int, default=100, help="Chebyshev degree timed in the configs[4] section")
    ap.add_argument("--cheb-batches", default="1,12", help="vectors per launch timed in the configs[4] section (divisors of 12)")
    ap.add_argument("--table-scale", type=float, default=1.0, help="scale the iteration counts of the kernel table")
    ap.add_argument("--l2-probe", action="store_true", help="only: read rate of qcd_redot on L2-resident vectors (L2 -> SM fabric)")
    return ap.parse_args()


def measured_peaks():
    """Roofline denominator: MEASURED_PEAKS.json (driver-written), else the fallback of
    /opt/skills/guides/B200_PROFILING.md (6.65 TB/s)."""
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    try:
        with open(p) as f:
            return float(json.load(f)["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)"
    except Exception:
        return 6650.0, "fallback (B200_PROFILING.md 6.65 TB/s)"


def workload_config(world):
    """`config` of the JSON line: the same dict for our arm and for the reference arm."""
    Vh = DIMS[0] * DIMS[1] * DIMS[2] * DIMS[3] // 2
    return {"workload": "even-odd Wilson-clover Dslash (Mhat_ee apply = 2 fused hop launches), 32^3x64, fp32, "
                        "12-real links, kappa 0.1355, csw 1.0, eps 0.5 (BASELINE.json configs[3] lattice, "
                        "north_star 70% target workload)",
            "dims": list(DIMS), "reconstruct": 12, "kappa": KAPPA, "csw": CSW, "eps": EPS,
            "parallelism": "replicas only (x%d)" % world,
            "l2": "inputs larger than L2 (gauge 403 MB + clover 604 MB per step) and the spinor buffers rotate over "
                  "3 distinct sets, so no launch finds its operands left in L2 by the previous one",
            "flop_per_step": step_flops(Vh), "gauge_recipe": "32^3x16 block of the configs[0] recipe tiled 4x in t"}


def step_flops(Vh, clover=True):
    return 2.0 * HOP_FLOP * Vh + (2.0 * CLOVER_FLOP * Vh if clover else 0.0)


class ClockSampler(threading.Thread):
    """Samples SM clock and throttle reasons with NVML while the timed region runs."""

    def __init__(self, index=0, period=0.02):
        super().__init__(daemon=True)
        self.index, self.period = index, period
        self.samples, self.reasons = [], set()
        self.max_mhz = None
        self._stop_evt = threading.Event()
        self.ok = False
        try:
            import pynvml
            pynvml.nvmlInit()
            self.nv = pynvml
            self.h = pynvml.nvmlDeviceGetHandleByIndex(index)
            self.max_mhz = pynvml.nvmlDeviceGetMaxClockInfo(self.h, pynvml.NVML_CLOCK_SM)
            self.ok = True
        except Exception:
            self.ok = False

    _NAMES = {0x1: "gpu_idle", 0x2: "applications_clocks_setting", 0x4: "sw_power_cap", 0x8: "hw_slowdown",
              0x10: "sync_boost", 0x20: "sw_thermal_slowdown", 0x40: "hw_thermal_slowdown",
              0x80: "hw_power_brake_slowdown", 0x100: "display_clock_setting"}

    def run(self):
        if not self.ok:
            return
        nv = self.nv
        while not self._stop_evt.is_set():
            try:
                self.samples.append(nv.nvmlDeviceGetClockInfo(self.h, nv.NVML_CLOCK_SM))
                try:
                    r = nv.nvmlDeviceGetCurrentClocksEventReasons(self.h)
                except Exception:
                    r = nv.nvmlDeviceGetCurrentClocksThrottleReasons(self.h)
                for bit, name in self._NAMES.items():
                    if r & bit and name != "gpu_idle":
                        self.reasons.add(name)
            except Exception:
                pass
            time.sleep(self.period)

    def stop(self):
        self._stop_evt.set()
        if self.is_alive():
            self.join(timeout=2)
        s = sorted(self.samples)
        return {"sm_mhz": (s[len(s) // 2] if s else None), "sm_max_mhz": self.max_mhz,
                "reasons": sorted(self.reasons), "samples": len(s)}


# ---------------------------------------------------------------------------------------
# CPU oracle leg (the only place bench.py executes oracle/): cpu_baseline and --impl reference
# ---------------------------------------------------------------------------------------
class OracleWorkload:
    """The oracle's Mhat_ee apply, as it stands, on a bounded sample of the workload: the
    16^3 x 32 lattice (1/16 of the 32^3 x 64 sites; same recipe, kappa, csw)."""

    sample = "Mhat_ee apply (oracle apply_M mode 0, fp64) on a 16^3x32 lattice = 1/16 of the 32^3x64 sites, same recipe"

    def __init__(self):
        import numpy as np
        from oracle import oracle as orc
        from paper_2001_05706_b200 import inputs
        self.orc, self.dims = orc, SMALL_DIMS
        self.U = inputs.gauge_field(self.dims, EPS, 0)
        F = orc.field_strength(self.U, self.dims)
        self.A = orc.clover_matrix(F, self.dims, KAPPA * CSW)
        self.Ainv = orc.invert_12(self.A)
        par = orc.parity_mask_array(self.dims)[..., None, None, None]
        self.psi = inputs.spinor_field(self.dims, 0, 0) * (par == 0)
        self.Vh = int(np.prod(self.dims)) // 2
        self.cores = orc.num_threads()

    def step(self):
        return self.orc.apply_M(self.psi, self.U, self.dims, KAPPA, self.A, self.Ainv, -1, 0, False)

    def time_steps(self, steps, warmup):
        for _ in range(warmup):
            self.step()
        t0 = time.perf_counter()
        for _ in range(steps):
            self.step()
        dt = (time.perf_counter() - t0) / max(steps, 1)
        return dt, step_flops(self.Vh) / dt * 1e-9


def cpu_baseline(budget_s=15.0):
    w = OracleWorkload()
    dt1, _ = w.time_steps(1, 1)
    n = max(1, min(200, int(budget_s / max(dt1, 1e-6))))
    dt, gf = w.time_steps(n, 0)
    return {"value": gf, "unit": UNIT, "cores": w.cores, "kind": "oracle", "sample": w.sample,
            "ms_per_step_on_sample": dt * 1e3}


def run_reference(args):
    """The reference arm of this tier is the oracle as it stands, on the host cores: same metric,
    unit and `config` as our arm, each step a bounded sample of that workload (OracleWorkload.sample).
    Under torchrun rank 0 alone runs and prints it."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    w = OracleWorkload()
    steps, warm = max(1, args.steps), max(0, args.warmup)
    dt, gf = w.time_steps(steps, warm)
    line = {
        "impl": "reference", "metric": METRIC, "value": gf, "unit": UNIT, "n_gpus": args.gpus, "steps": steps,
        "warmup": warm, "ms_per_step": dt * 1e3, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
        "dtype": "f64", "data": "synthetic", "config": workload_config(max(1, args.gpus)),
        "cpu_baseline": {"value": gf, "unit": UNIT, "cores": w.cores, "kind": "oracle", "sample": w.sample},
        "e2e": {"value": gf, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    print(json.dumps(line))


# ---------------------------------------------------------------------------------------
# CUDA arm
# ---------------------------------------------------------------------------------------
NSETS = 3   # distinct operand sets the timed loops rotate over (a 101 MB spinor block fits
            # the 126 MB L2, so back-to-back launches on ONE set find part of their input still cached)


def gpu_time_ms(fn, iters, warm=3):
    """Average device time of fn(i) in ms: CUDA events on the launching stream (the ctx is
    bound to torch's current stream), after warm-up, synchronised on both sides.  fn gets the
    iteration number and picks operand set i % NSETS."""
    import torch
    iters = max(1, int(iters * TABLE_SCALE))
    for i in range(warm if TABLE_SCALE >= 1.0 else 1):
        fn(i)
    torch.cuda.synchronize()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record()
    for i in range(iters):
        fn(i)
    e1.record()
    e1.synchronize()
    return e0.elapsed_time(e1) / iters


def sets_of(t, n=NSETS):
    """n distinct copies of a device tensor"""
    return [t.clone() for _ in range(n)]


def build_workload(c, dims, want_hi):
    """Seeded synthetic fields on the device.  Links: configs[0] recipe with eps = 0.5 on a
    (X,Y,Z,16) block repeated along t (inputs.tiled_gauge_field); source: N(0,1)."""
    import torch
    from paper_2001_05706_b200 import inputs
    U = inputs.tiled_gauge_field(dims, EPS, 0, 16)
    dU = torch.from_numpy(U).cuda()
    del U
    w = {"dims": dims}
    g_hi = c.gauge_load(dU, dims, 8, 18, -1)
    w["g32"] = c.gauge_load(dU, dims, 4, 12, -1)
    w["c32"] = c.clover_build(g_hi, KAPPA, CSW, 4)          # fp64 arithmetic, fp32 storage (S15)
    if want_hi:
        w["g32_18"] = c.gauge_load(dU, dims, 4, 18, -1)
        w["g64"] = g_hi
        w["g64_12"] = c.gauge_load(dU, dims, 8, 12, -1)
        w["c64"] = c.clover_build(g_hi, KAPPA, CSW, 8)
        w["g16"] = c.gauge_load(dU, dims, 2, 12, -1)           # 16-bit storage (reading H1)
        w["c16"] = c.clover_build(g_hi, KAPPA, CSW, 2)
    del dU
    psi = torch.from_numpy(inputs.spinor_field(dims, 0, 0))
    w["psi64"] = c.spinor_pack(psi.cuda(), dims) if want_hi else None
    w["psi32"] = c.spinor_pack(psi.float().cuda(), dims)
    torch.cuda.synchronize()
    return w


def traffic_from_profile():
    """dram__bytes_read.sum + dram__bytes_write.sum per launch of the dominant kernel, from the
    committed ncu --set full capture (profiles/traffic.csv); None if there is no capture."""
    import csv
    try:
        with open(os.path.join(ROOT, "profiles", "traffic.csv")) as f:
            for row in csv.DictReader(f):
                if row["kernel"] == "hop_clover_fp32_12":
                    return float(row["bytes_per_launch"])
    except Exception:
        pass
    return None


def kernel_table(c, w, peak):
    """Every other kernel of the path against the HBM roofline (SURVEY.md 8(d) bytes/site)."""
    import torch
    dims = w["dims"]
    Vh = dims[0] * dims[1] * dims[2] * dims[3] // 2
    out = {}

    def row(name, ms, bytes_per_site, flop_per_site):
        gbs = bytes_per_site * Vh / (ms * 1e-3) * 1e-9
        out[name] = {"us": round(ms * 1e3, 2), "GB/s": round(gbs, 1), "frac": round(gbs / peak, 4),
                     "GFLOP/s": round(flop_per_site * Vh / (ms * 1e-3) * 1e-9, 1), "B/site": bytes_per_site}

    h = Vh * 24
    R = range(NSETS)
    a32, z32 = sets_of(w["psi32"][:h]), sets_of(w["psi32"][h:])
    b32 = [torch.empty_like(a32[0]) for _ in R]
    row("hop_fp32_12", gpu_time_ms(lambda i: c.hop(b32[i % NSETS], z32[i % NSETS], w["g32"], 0), 60), 576, 1320)
    row("hop_fp32_18", gpu_time_ms(lambda i: c.hop(b32[i % NSETS], z32[i % NSETS], w["g32_18"], 0), 60), 768, 1320)
    row("hop_xpay_fp32_12", gpu_time_ms(lambda i: c.hop_xpay(b32[i % NSETS], z32[i % NSETS], a32[i % NSETS], 1.0, -KAPPA, w["g32"], 0), 60), 672, 1320)
    a64, z64 = sets_of(w["psi64"][:h]), sets_of(w["psi64"][h:])
    b64 = [torch.empty_like(a64[0]) for _ in R]
    tmp64 = [torch.empty_like(a64[0]) for _ in R]
    row("hop_fp64_18", gpu_time_ms(lambda i: c.hop(b64[i % NSETS], z64[i % NSETS], w["g64"], 0), 21), 1536, 1320)
    ms = gpu_time_ms(lambda i: c.dslash_ex(b64[i % NSETS], a64[i % NSETS], w["g64"], w["c64"], KAPPA, CSW, 0, 0, tmp64[i % NSETS]), 21)
    row("Mhat_clover_fp64_18 (2 launches)", ms, 2 * 1536 + 2 * 576 + 192, 2 * 1320 + 2 * 504)
    row("hop_fp64_12", gpu_time_ms(lambda i: c.hop(b64[i % NSETS], z64[i % NSETS], w["g64_12"], 0), 21), 1152, 1320)
    ms = gpu_time_ms(lambda i: c.dslash_ex(b64[i % NSETS], a64[i % NSETS], w["g64_12"], w["c64"], KAPPA, CSW, 0, 0, tmp64[i % NSETS]), 21)
    row("Mhat_clover_fp64_12 (2 launches)", ms, 2 * 1152 + 2 * 576 + 192, 2 * 1320 + 2 * 504)
    del a64, z64, b64, tmp64
    # 16-bit storage (reading H1): 52 B spinor site, 24 B link, 148 B clover site
    hb = Vh * 52
    ph = sets_of(c.spinor_to_half(w["psi32"], dims, 2)[:hb])
    o16, t16 = [c.empty(hb) for _ in R], [c.empty(hb) for _ in R]
    ms = gpu_time_ms(lambda i: c.dslash_half(o16[i % NSETS], 2, ph[i % NSETS], w["g16"], None, KAPPA, 0.0, 0, 0, t16[i % NSETS]), 60)
    row("Mhat_wilson_q16_12 (2 launches: hop, hop+xpay)", ms, 2 * (52 + 192 + 52) + 52, 2 * 1320)
    ms = gpu_time_ms(lambda i: c.dslash_half(o16[i % NSETS], 2, ph[i % NSETS], w["g16"], w["c16"], KAPPA, CSW, 0, 0, t16[i % NSETS]), 60)
    row("Mhat_clover_q16_12 (2 launches)", ms, 2 * (52 + 192 + 148 + 52) + 52, 2 * 1320 + 2 * 504)
    del ph, o16, t16
    # fused BLAS-1, one-parity vectors (100 MB each in fp32); NSETS sets of 4 distinct arrays
    X, Y, P, Q = ([torch.randn(h, device="cuda", dtype=torch.float32) for _ in R] for _ in range(4))
    row("axpy_fp32", gpu_time_ms(lambda i: c.axpy(1e-3, X[i % NSETS], Y[i % NSETS]), 60), 288, 48)
    row("xpay_fp32", gpu_time_ms(lambda i: c.xpay(X[i % NSETS], 0.5, Y[i % NSETS]), 60), 288, 48)
    row("norm2_fp32", gpu_time_ms(lambda i: c.norm2(X[i % NSETS], fetch=False), 60), 96, 48)
    row("redot_fp32", gpu_time_ms(lambda i: c.redot(X[i % NSETS], Y[i % NSETS], fetch=False), 60), 192, 96)
    row("cg_update_fp32", gpu_time_ms(lambda i: c.cg_update(1e-6, P[i % NSETS], Q[i % NSETS], X[i % NSETS], Y[i % NSETS], fetch=False), 60), 576, 144)
    X, Y, P, Q = ([t.double() for t in v] for v in (X, Y, P, Q))
    row("cg_update_fp64", gpu_time_ms(lambda i: c.cg_update(1e-6, P[i % NSETS], Q[i % NSETS], X[i % NSETS], Y[i % NSETS], fetch=False), 21), 1152, 144)
    row("redot_fp64", gpu_time_ms(lambda i: c.redot(X[i % NSETS], Y[i % NSETS], fetch=False), 21), 384, 96)
    row("norm2_fp64", gpu_time_ms(lambda i: c.norm2(X[i % NSETS], fetch=False), 21), 192, 48)
    row("axpy_fp64", gpu_time_ms(lambda i: c.axpy(1e-3, X[i % NSETS], Y[i % NSETS]), 21), 576, 48)
    return out


def solver_table(c, w):
    """CG seconds to 1e-10 (BASELINE.json metric, second half): even-odd clover, 32^3x64."""
    import torch
    from paper_2001_05706_b200 import inputs
    dims = w["dims"]
    Vh = dims[0] * dims[1] * dims[2] * dims[3] // 2
    h = Vh * 24
    b = c.spinor_pack(torch.from_numpy(inputs.spinor_field(dims, 0, 1)).cuda(), dims)[:h].clone()
    x = torch.empty_like(b)
    out = {}
    c.ensure_workspace(c.workspace_bytes(dims, 8))
    # fp64 operator with 18-real links (reading S15) and with 12-real links (row 2 rebuilt in fp64: same iterations and
    # residuals, 25 % fewer link bytes: the fp64 12-real hop is the faster one on B200)
    for name, lo, ghi in (("cg_fp64_18", 0, "g64"), ("cg_fp64_12", 0, "g64_12"), ("mixed_cg_fp32_12/fp64_18", 1, "g64"),
                          ("mixed_cg_fp32_12/fp64_12", 1, "g64_12"), ("mixed_cg_q16_12/fp64_18", 2, "g64")):
        if lo == 2:
            c.set_operator(w[ghi], w["g16"], w["c64"], w["c16"], KAPPA, CSW, 0, 0.1)
        elif lo:
            c.set_operator(w[ghi], w["g32"], w["c64"], w["c32"], KAPPA, CSW, 0, 0.1)
        else:
            c.set_operator(w[ghi], None, w["c64"], None, KAPPA, CSW, 0)
        c.cg_solve(x, b, 1e-10, 5000)                      # warm-up solve
        rc, st = c.cg_solve(x, b, 1e-10, 5000)
        out[name] = {"seconds": round(st.seconds, 5), "iters": st.iters, "reliable_updates": st.reliable_updates,
                     "r_true": st.r_true, "rc": rc, "GFLOP/s": round(st.flops / st.seconds * 1e-9, 1),
                     "ms_per_iter": round(st.seconds / max(st.iters, 1) * 1e3, 4)}
    # multi-shift CG: 4 shifted systems for the price of one N apply per iteration
    shifts = [0.0, 0.01, 0.1, 1.0]
    xs = torch.empty(len(shifts) * h, dtype=b.dtype, device="cuda")
    c.set_operator(w["g64"], None, w["c64"], None, KAPPA, CSW, 0)
    c.ensure_workspace((4 + len(shifts)) * h * 8)
    c.cg_multishift(xs, b, shifts, 1e-10, 5000)
    rc, st, rts = c.cg_multishift(xs, b, shifts, 1e-10, 5000)
    out["multishift_cg_fp64_18 (4 shifts)"] = {"seconds": round(st.seconds, 5), "iters": st.iters, "rc": rc, "shifts": shifts,
                                               "r_true_max": max(rts), "ms_per_iter": round(st.seconds / max(st.iters, 1) * 1e3, 4)}
    return out


def cheb_batches(args):
    nbs = tuple(int(v) for v in args.cheb_batches.split(","))
    assert all(nb >= 1 and 12 % nb == 0 for nb in nbs), "--cheb-batches: divisors of 12"
    return nbs


def config_table(c, peak, config4, only4=False, cheb_degree=100, cheb_batches=(1, 12)):
    """The other BASELINE.json configs at their full sizes (parity for each is in tests/)."""
    import torch
    from paper_2001_05706_b200 import inputs
    out = {}
    if not only4:
        # configs[1]: 16^3x32 fp32 even-odd Wilson, kappa 0.137, 18- and 12-real; single apply + 100-loop.
        dims, kappa = (16, 16, 16, 32), 0.137
        Vh = 16 * 16 * 16 * 32 // 2
        h = Vh * 24
        dU = torch.from_numpy(inputs.gauge_field(dims, EPS, 0)).cuda()
        pin = c.spinor_pack(torch.from_numpy(inputs.spinor_field(dims, 0, 0)).float().cuda(), dims)
        src, dst, tmp = pin[:h].clone(), torch.empty_like(pin[:h]), torch.empty_like(pin[:h])
        from paper_2001_05706_b200 import qcd
        gs = torch.cuda.Stream()
        cgx = qcd.Context(torch.cuda.current_device(), stream=gs)   # a ctx on a capturable side stream
        for rec in (18, 12):
            g = c.gauge_load(dU, dims, 4, rec, -1)
            fn = lambda i=0: c.dslash_ex(dst, src, g, None, kappa, 0.0, 0, 0, tmp)
            loop_ms = gpu_time_ms(fn, 100)
            # the same 100-apply loop captured once in a CUDA graph and replayed (SURVEY 8(d) caveat i)
            gs.wait_stream(torch.cuda.current_stream())
            with torch.cuda.stream(gs):
                gg = cgx.gauge_load(dU, dims, 4, rec, -1)
                cgx.dslash_ex(dst, src, gg, None, kappa, 0.0, 0, 0, tmp)
            gs.synchronize()
            graph = torch.cuda.CUDAGraph()
            with torch.cuda.graph(graph, stream=gs):
                for _ in range(100):
                    cgx.dslash_ex(dst, src, gg, None, kappa, 0.0, 0, 0, tmp)
            graph.replay()
            torch.cuda.synchronize()
            g0, g1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            g0.record()
            for _ in range(5):
                graph.replay()
            g1.record(); g1.synchronize()
            graph_ms = g0.elapsed_time(g1) / 500.0
            torch.cuda.synchronize()
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            e0.record(); fn(); e1.record(); e1.synchronize()
            flop = 2 * HOP_FLOP * Vh
            byts = (2 * (48 + 8 * rec) + 24) * 4 * Vh
            out["config1_wilson_eo_16x32_fp32_%d" % rec] = {
                "single_apply_us": round(e0.elapsed_time(e1) * 1e3, 2), "loop100_us_per_apply": round(loop_ms * 1e3, 2),
                "graph100_us_per_apply": round(graph_ms * 1e3, 2),
                "GFLOP/s": round(flop / (loop_ms * 1e-3) * 1e-9, 1), "GB/s": round(byts / (loop_ms * 1e-3) * 1e-9, 1),
                "frac": round(byts / (loop_ms * 1e-3) * 1e-9 / peak, 4),
                "note": "L2-resident (38-50 MB working set): the HBM fraction is not a roofline statement here"}
        del dU
        # configs[2]: 24^3x64 fp64 Wilson-clover CG, kappa 0.135, csw 1, tol 1e-10, maxiter 5000.
        dims, kappa = (24, 24, 24, 64), 0.135
        Vh = 24 * 24 * 24 * 64 // 2
        h = Vh * 24
        dU = torch.from_numpy(inputs.tiled_gauge_field(dims, EPS, 0, 16)).cuda()
        g = c.gauge_load(dU, dims, 8, 18, -1)
        g12 = c.gauge_load(dU, dims, 8, 12, -1)
        del dU
        cl = c.clover_build(g, kappa, CSW, 8)
        b = c.spinor_pack(torch.from_numpy(inputs.spinor_field(dims, 0, 1)).cuda(), dims)
        c.ensure_workspace(c.workspace_bytes(dims, 8))
        for name, mode, gg in (("config2_clover_cg_24x64_fp64_evenodd", 0, g), ("config2_clover_cg_24x64_fp64_full", 2, g),
                               ("config2_clover_cg_24x64_fp64_evenodd_12real", 0, g12), ("config2_clover_cg_24x64_fp64_full_12real", 2, g12)):
            c.set_operator(gg, None, cl, None, kappa, CSW, mode)
            bb = b[:h].clone() if mode == 0 else b
            x = torch.empty_like(bb)
            c.cg_solve(x, bb, 1e-10, 5000)
            rc, st = c.cg_solve(x, bb, 1e-10, 5000)
            out[name] = {"seconds": round(st.seconds, 5), "iters": st.iters, "r_true": st.r_true, "rc": rc,
                         "GFLOP/s": round(st.flops / st.seconds * 1e-9, 1), "ms_per_iter": round(st.seconds / max(st.iters, 1) * 1e3, 4)}
        del g, g12, cl, b
    if config4:
        # configs[4]: degree-100 Chebyshev of H_W (kappa 0.2) on 12 Gaussian vectors, 48^3x96 fp32.
        dims, kappa, scale, nvec = (48, 48, 48, 96), 0.2, 2.6, 12
        V = 48 * 48 * 48 * 96
        dU = torch.from_numpy(inputs.tiled_gauge_field(dims, EPS, 0, 8).astype("float32")).cuda()
        g = c.gauge_load(dU, dims, 4, 12, -1)
        del dU
        coeff = inputs.chebyshev_sign_coefficients(100)[:cheb_degree + 1]
        res = {}
        for nb in cheb_batches:
            v = torch.randn(nb * V * 24, device="cuda", dtype=torch.float32)
            y = torch.empty_like(v)
            c.set_workspace(None)
            c.ensure_workspace(2 * nb * V * 24 * 4)
            c.cheb_apply_multi(y, v, nb, g, kappa, coeff[:4], scale)
            torch.cuda.synchronize()
            sampler = ClockSampler(torch.cuda.current_device())
            sampler.start()
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            e0.record()
            for _ in range(nvec // nb):
                c.cheb_apply_multi(y, v, nb, g, kappa, coeff, scale)
            e1.record(); e1.synchronize()
            clk = sampler.stop()
            sec = e0.elapsed_time(e1) * 1e-3
            per_sv = 480.0 + 384.0 / nb       # in + z + b_{k+2} + v + out = 5 x 96 B, links 384 B / nb
            byts = per_sv * (V // 2) * nvec * cheb_degree * 2
            res["%d vector(s) per launch" % nb] = {
                "seconds_12vec_deg%d" % cheb_degree: round(sec, 4),
                "GFLOP/s": round(HOP_FLOP * (V // 2) * nvec * 2 * cheb_degree / sec * 1e-9, 1),
                "GB/s": round(byts / sec * 1e-9, 1), "frac": round(byts / sec * 1e-9 / peak, 4), "B/site-vector": per_sv, "clocks": clk}
            if nb == nvec:
                # plain multi-rhs Wilson operator (qcd_wilson_multi): in + z + out per site-vector, links once per block
                ms = gpu_time_ms(lambda i: c.wilson_multi(y, v, nb, g, kappa, True), 10)
                per = 288.0 + 384.0 / nb
                res["qcd_wilson_multi, %d vectors (2 launches)" % nb] = {
                    "ms": round(ms, 3), "GFLOP/s": round(HOP_FLOP * V * nb / (ms * 1e-3) * 1e-9, 1),
                    "GB/s": round(per * V * nb / (ms * 1e-3) * 1e-9, 1), "frac": round(per * V * nb / (ms * 1e-3) * 1e-9 / peak, 4),
                    "B/site-vector": per}
            del v, y
        res["note"] = "Clenshaw recurrence, gamma5 and the coefficient term fused in the hop epilogue (2 launches per degree)"
        out["config4_chebyshev_48x96_fp32_12vec_deg%d" % cheb_degree] = res
    return out


def l2_probe():
    """Read rate of a pure streaming kernel (qcd_redot, fp64) on vectors that stay resident in the 126 MB L2:
    what the L2 -> SM fabric delivers on this part, for profiles/hop_cheb_mrhs_r2.md.  Launch overhead is in
    the per-launch time, so the rate is read off the increments between sizes."""
    import torch
    from paper_2001_05706_b200 import build, qcd
    build.build()
    c = qcd.Context(0)
    sampler = ClockSampler(0)
    sampler.start()
    rows = []
    for mb in (16, 32, 48, 64, 80, 96, 112, 160, 1024):
        n = mb * (1 << 20) // 16
        x = torch.randn(n, device="cuda", dtype=torch.float64)
        y = torch.randn(n, device="cuda", dtype=torch.float64)
        for _ in range(50):
            c.redot(x, y, fetch=False)
        torch.cuda.synchronize()
        best = 1e9
        for _ in range(3):
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            e0.record()
            for _ in range(1000):
                c.redot(x, y, fetch=False)
            e1.record(); e1.synchronize()
            best = min(best, e0.elapsed_time(e1))          # us per launch (1000 launches, ms total)
        rows.append({"MB": mb, "us_per_launch": round(best, 2), "TB/s_incl_launch": round(mb * 1.048576 / best, 2)})
        del x, y
    print(json.dumps({"l2_probe": rows, "clocks": sampler.stop()}))


def max_over_ranks(ms, device="cuda"):
    """Multi-GPU timing rule: every rank contributes its device time, the job's time is the MAX
    (replicas only: no data-path collective, this all-reduce is outside the timed region)."""
    import torch
    import torch.distributed as dist
    if not (dist.is_available() and dist.is_initialized()) or dist.get_world_size() == 1:
        return float(ms)
    t = torch.tensor([float(ms)], device=device, dtype=torch.float64)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def job_value(world, flop_per_step_per_rank, ms_step):
    """Whole-job throughput of `world` independent replicas (weak scaling)."""
    return world * flop_per_step_per_rank / (ms_step * 1e-3) * 1e-9


def run_ours(args):
    import torch
    import torch.distributed as dist
    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device (the product path has no CPU fallback)")
    torch.cuda.set_device(local)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))

    from paper_2001_05706_b200 import build
    if rank == 0:
        build.build()
    if world > 1:
        dist.barrier()
    from paper_2001_05706_b200 import qcd
    c = qcd.Context(local)
    peak, peak_src = measured_peaks()
    full = (not args.quick) and rank == 0 and not args.config4_only
    w = build_workload(c, DIMS, want_hi=full)
    dims = DIMS
    Vh = dims[0] * dims[1] * dims[2] * dims[3] // 2
    h = Vh * 24
    srcs = sets_of(w["psi32"][:h])
    dsts = [torch.empty_like(srcs[0]) for _ in range(NSETS)]
    tmps = [torch.empty_like(srcs[0]) for _ in range(NSETS)]
    src = srcs[0]
    g, cl = w["g32"], w["c32"]

    def step(i=0):
        k = i % NSETS
        c.dslash_ex(dsts[k], srcs[k], g, cl, KAPPA, CSW, 0, 0, tmps[k])

    # ---- timed region: W warm-up steps, then exactly K steps between barrier + synchronize
    for i in range(max(args.warmup, 3)):
        step(i)
    torch.cuda.synchronize()
    if world > 1:
        dist.barrier()
    sampler = ClockSampler(local)
    sampler.start()
    n0 = c.launch_count()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    torch.cuda.synchronize()
    e0.record()
    for i in range(args.steps):
        step(i)
    e1.record()
    torch.cuda.synchronize()
    ms_total = e0.elapsed_time(e1)
    launches = c.launch_count() - n0
    clocks = sampler.stop()
    if world > 1:
        dist.barrier()
    ms_total = max_over_ranks(ms_total)
    ms_step = ms_total / args.steps
    value = job_value(world, step_flops(Vh), ms_step)

    # ---- roofline of the dominant kernel (hop_kernel<float,12,*,CLOVER_*>): two launches per
    # step, algorithmic bytes 864 (clover-inverse epilogue) and 960 (clover + xpay) per site
    bytes_launch = 0.5 * (864 + 960) * Vh
    ms_launch = ms_step / 2.0
    achieved = bytes_launch / (ms_launch * 1e-3) * 1e-9
    roofline = {"bound": "hbm", "achieved": round(achieved, 1), "peak": peak, "unit": "GB/s",
                "frac": round(achieved / peak, 4), "traffic": traffic_from_profile(), "peak_source": peak_src,
                "kernel": "hop_kernel<float,12,0,CLOVER_OUT|CLOVER_Z>", "bytes_per_launch": bytes_launch,
                "us_per_launch": round(ms_launch * 1e3, 2)}

    # ---- end to end: HOST buffers through the C ABI, H2D + Mhat + D2H for every step inside the
    # timed region.  qcd_dslash_host_batch pipelines the steps (H2D of step i+1, operator on step i,
    # D2H of step i-1 overlap); qcd_dslash_host is the same thing one synchronous call per step.
    blk_bytes = h * 4
    e2e_steps = max(4, min(16, args.steps))
    c.ensure_workspace(max(5 * blk_bytes, c._ws.numel() if c._ws is not None else 0))
    hin = torch.empty(e2e_steps * h, dtype=torch.float32).pin_memory()
    hout = torch.empty(e2e_steps * h, dtype=torch.float32).pin_memory()
    hsrc = src.cpu()
    for i in range(e2e_steps):
        hin[i * h:(i + 1) * h].copy_(hsrc)
    del hsrc
    c.dslash_host_batch(hout, hin, e2e_steps, g, cl, KAPPA, CSW, 0, 0)        # warm-up (creates the copy streams)
    torch.cuda.synchronize()
    # the host side of PCIe is shared with whatever else runs on the box: three timed calls of e2e_steps steps
    # each, the median reported (all three kept in the line)
    e2e_reps = []
    for _ in range(3):
        t0 = time.perf_counter()
        e0.record()
        c.dslash_host_batch(hout, hin, e2e_steps, g, cl, KAPPA, CSW, 0, 0)
        e1.record()
        torch.cuda.synchronize()
        e2e_reps.append(max_over_ranks(max(e0.elapsed_time(e1), (time.perf_counter() - t0) * 1e3) / e2e_steps))
    e2e_ms = sorted(e2e_reps)[1]
    for _ in range(2):
        c.dslash_host(hout[:h], hin[:h], g, cl, KAPPA, CSW, 0, 0)
    torch.cuda.synchronize()
    t0 = time.perf_counter()
    for _ in range(e2e_steps):
        c.dslash_host(hout[:h], hin[:h], g, cl, KAPPA, CSW, 0, 0)
    torch.cuda.synchronize()
    sync_ms = max_over_ranks((time.perf_counter() - t0) * 1e3 / e2e_steps)
    e2e = {"value": round(job_value(world, step_flops(Vh), e2e_ms), 1), "unit": UNIT,
           "h2d_bytes_per_step": blk_bytes, "d2h_bytes_per_step": blk_bytes, "ms_per_step": round(e2e_ms, 4),
           "steps": e2e_steps, "ms_per_step_of_each_timed_call": [round(v, 4) for v in e2e_reps],
           "call": "qcd_dslash_host_batch (pipelined H2D / Mhat / D2H, pinned host buffers)",
           "one_call_per_step": {"value": round(job_value(world, step_flops(Vh), sync_ms), 1), "ms_per_step": round(sync_ms, 4),
                                 "call": "qcd_dslash_host"}}
    del hin, hout

    if rank != 0:
        if world > 1:
            dist.barrier()
            dist.destroy_process_group()
        return
    line = {
        "metric": METRIC, "value": round(value, 1), "unit": UNIT, "n_gpus": world, "steps": args.steps,
        "warmup": max(args.warmup, 3), "ms_per_step": round(ms_step, 5), "higher_is_better": True,
        "scaling": "weak", "vs_baseline": None, "dtype": "f32", "data": "synthetic",
        "config": workload_config(world),
        "clocks": clocks, "e2e": e2e, "gpu_launches": int(launches), "roofline": roofline,
    }
    if not args.no_cpu_baseline:
        line["cpu_baseline"] = cpu_baseline()
    if full and args.solvers_only:
        line["cg"] = solver_table(c, w)
    elif full:
        line["kernels"] = kernel_table(c, w, peak)
        if not args.no_solvers:
            line["cg"] = solver_table(c, w)
            del w
            torch.cuda.empty_cache()
            line["configs"] = config_table(c, peak, not args.no_config4, cheb_degree=args.cheb_degree, cheb_batches=cheb_batches(args))
    if args.config4_only and rank == 0:
        del w
        torch.cuda.empty_cache()
        line["configs"] = config_table(c, peak, True, only4=True, cheb_degree=args.cheb_degree, cheb_batches=cheb_batches(args))
    print(json.dumps(line))
    if world > 1:
        dist.barrier()
        dist.destroy_process_group()


def spawn_replicas(args):
    """`python bench.py --gpus N` without a launcher: start the N ranks ourselves, the way the driver
    does (one process per GPU, torch.distributed.run on 127.0.0.1), and pass rank 0's JSON line through."""
    import socket
    import subprocess
    import torch
    have = torch.cuda.device_count()
    if have < args.gpus:
        raise SystemExit("bench.py: --gpus %d asked for, %d CUDA device(s) visible" % (args.gpus, have))
    with socket.socket() as sk:
        sk.bind(("127.0.0.1", 0))
        port = sk.getsockname()[1]
    raise SystemExit(subprocess.call(replica_command(args.gpus, port, sys.argv[1:])))


def replica_command(ngpus, port, argv):
    return [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node", str(ngpus),
            "--master-addr", "127.0.0.1", "--master-port", str(port), os.path.abspath(__file__)] + list(argv)


if __name__ == "__main__":
    a = parse_args()
    TABLE_SCALE = a.table_scale
    if a.l2_probe:
        l2_probe()
    elif a.impl == "reference":
        run_reference(a)
    elif a.gpus > 1 and "WORLD_SIZE" not in os.environ:
        spawn_replicas(a)
    else:
        run_ours(a)
