"""bench.py -- throughput of the STREAmS-2 hot path (RHS + RK3) on B200, in grid-point RK-step updates/s.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--config I] [--impl ours|reference]
    python -m torch.distributed.run --nnodes=1 --nproc-per-node N ... bench.py --gpus N ...

A "step" is one full low-storage RK3 step of the whole hot path over the whole grid: 3 x (ghost fill, sensor/mask,
interface flags, WENO fluxes of the flagged interfaces, fused convective x/y/z + viscous RHS + RK update + primitives
of the updated state) and the dt reduction.  value = grid points x K / device time of streams_step(K)
(= 1e8 / the paper's "grind time").  The workload is BASELINE.json configs[4], the largest single-GPU
configuration (640^3 periodic compressible turbulence, hybrid WENO, Sutherland viscosity; BASELINE.json's `metric` names
no config of its own and configs[4] is its "per-kernel roofline capture" run) unless --config says otherwise; the
timed region is repeated --repeats times from the same state, `value` is the median, the best is reported beside it.
N > 1: the path is single-GPU by design (north_star); ranks run independent replicas with different
seeds and no data-path collective ("replicas only"), value = sum over ranks / max time.

One JSON line on stdout from rank 0; keys as the driver's contract plus `roofline` and `cpu_baseline`.
`--impl reference` times the CPU oracle (oracle/, the only "reference" that exists for this paper) on the
host cores on the same workload and prints the same line with "impl": "reference".
"""
from __future__ import annotations

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

import numpy as np  # noqa: E402

import workloads as W  # noqa: E402

METRIC = "fp64 grid-point RK-step updates/sec"
UNIT = "point-steps/s"


def load_peaks():
    """Measured roofline denominators (driver-written); fallback per B200_PROFILING.md."""
    path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(path):
        with open(path) as f:
            return float(json.load(f)["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)"
    return 6650.0, "fallback (B200_PROFILING.md 6.65 TB/s)"


def make_case(index: int, seed_offset: int = 0, cube: int = 256):
    """BASELINE.json configs[index] with the rank's seed (replicas differ only by seed: base + 100 * rank,
    paper_2304_05494_b200.replicas.replica_seed)."""
    if index == 0:
        return W.config(0)
    if index == 1:
        return W.isotropic_turbulence(n=128, mach_t=0.6, k0=4.0, kmax=32, seed=1 + 100 * seed_offset, nsteps=50,
                                      name="cfg1_iso_128")
    if index == 2:
        return W.channel(256, 192, 128, seed=2 + 100 * seed_offset, nsteps=50)
    if index == 3:
        return W.boundary_layer(1024, 256, 256, seed=3 + 100 * seed_offset, nsteps=20)
    if index == 4:
        return W.isotropic_turbulence(n=640, mach_t=0.8, k0=8.0, kmax=64, seed=4 + 100 * seed_offset, nsteps=10,
                                      name="cfg4_iso_640")
    if index == 5:   # SURVEY 8(d) "opt": the paper's own grid shape, not divisible by any tile
        return W.isotropic_turbulence(nx=420, ny=250, nz=320, mach_t=0.6, k0=4.0, kmax=32, seed=5 + 100 * seed_offset,
                                      nsteps=20, name="opt_iso_420x250x320")
    if index == 6:   # size sweep (Fig. 5: throughput against the number of grid points): --cube N
        return W.isotropic_turbulence(n=cube, mach_t=0.6, k0=4.0, kmax=min(32, cube // 4), seed=6 + 100 * seed_offset,
                                      nsteps=20, name=f"sweep_iso_{cube}")
    raise SystemExit(f"unknown config {index}")


WORKLOAD_TEXT = {
    0: "configs[0]: inviscid Taylor-Green vortex 32^3 periodic, central L=3, CFL 0.5",
    1: "configs[1]: viscous decaying compressible isotropic turbulence 128^3 periodic, Mach_t 0.6, k0=4, "
       "Sutherland, Pr 0.72, hybrid WENO5/central6 thr 0.2",
    2: "configs[2]: supersonic isothermal-wall channel 256x192x128, tanh-stretched y, hybrid",
    3: "configs[3]: supersonic flat-plate boundary-layer box 1024x256x256, stretched y, hybrid, seeded shocklets",
    4: "configs[4]: capacity run 640^3 periodic compressible turbulence Mach_t 0.8, k0=8, hybrid",
    5: "sweep grid 420x250x320 (the paper's grid shape, PAPER:355), periodic turbulence as configs[1]",
    6: "size sweep: N^3 periodic turbulence as configs[1] (--cube N)",
}


# ------------------------------------------------------------------------------------------------
# clocks during the timed region (B200_PROFILING.md "clocks line")
# ------------------------------------------------------------------------------------------------
class ClockSampler:
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, index: int):
        self.f = tempfile.NamedTemporaryFile("w+", suffix=".csv", delete=False)
        self.p = None
        try:
            self.p = subprocess.Popen(["nvidia-smi", f"--query-gpu={self.Q}", "--format=csv,noheader,nounits",
                                       "-lms", "100", "-i", str(index)], stdout=self.f, stderr=subprocess.DEVNULL)
        except OSError:
            self.p = None

    def stop(self):
        out = {"sm_mhz": None, "sm_max_mhz": None, "reasons": [], "samples": 0}
        if self.p is None:
            return out
        time.sleep(0.15)
        self.p.terminate()
        try:
            self.p.wait(timeout=5)
        except subprocess.TimeoutExpired:
            self.p.kill()
        self.f.flush()
        self.f.seek(0)
        sm, mx, pw, reasons = [], [], [], set()
        names = ("hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap")
        for line in self.f.read().splitlines():
            c = [x.strip() for x in line.split(",")]
            if len(c) < 7:
                continue
            try:
                sm.append(float(c[0])); mx.append(float(c[1])); pw.append(float(c[2]))
            except ValueError:
                continue
            for n, v in zip(names, c[3:7]):
                if v.lower().startswith("active"):
                    reasons.add(n)
        self.f.close()
        try:
            os.unlink(self.f.name)
        except OSError:
            pass
        if sm:
            out.update(sm_mhz=float(np.median(sm)), sm_max_mhz=float(max(mx)), power_w_max=float(max(pw)),
                       reasons=sorted(reasons), samples=len(sm))
        return out


# ------------------------------------------------------------------------------------------------
# algorithmic bytes per launch of each kernel class
# ------------------------------------------------------------------------------------------------
# fp64 instructions per unit of work: EXECUTED thread-level DFMA + DADD + DMUL (+ DSETP, MUFU.RCP64H) per node /
# padded node / flagged interface, orders 6/5/6, from the per-instruction execution counts of the ncu source page
# / the executed-instruction counters of profiles/r2_traffic_cfg4.md and profiles/r2_order_sweep.md (static SASS counts
# overstate kernels with branches: the IEEE-divide slow paths and the wall branch of fill_prim are rarely taken)
FP64_INST = {"rhs_main_cv": 463, "rhs_main_c": 200, "rhs_main_v": 265, "rhs_main_0": 15, "rhs_corr": 5, "corr_gather": 30,
             "weno_hybrid": 868, "weno_dense": 778, "fill_prim": 120, "fill_prim_dt": 50, "sensor": 97,
             "prims": 60}      # prims: cons -> prim of the updated node in the fused RHS epilogue (shared reciprocal, no IEEE divide)
FP64_LANES_PER_SM, N_SM = 64, 148       # B200: 64 fp64 FMA lanes per SM (37.2 TFLOP/s at 1965 MHz), 148 SMs


def case_is_hybrid(case):
    return case.flux_mode == 2


def work_model(case, act):
    """Per launch of each kernel class, averaged over the three RK stages of a step:
    bytes = what the method must move (every input field read once, every output written once, no halo
    re-reads), inst = fp64 thread-instructions.  act: mean fractions of N per sensor evaluation
    {"shock": nodes next to a flagged interface, "iface": flagged interfaces, all three directions}."""
    ng = 3
    N = case.npoints
    Np = (case.nx + 2 * ng) * (case.ny + 2 * ng) * (case.nz + 2 * ng)
    visc = case.visc_law != W.VISC_NONE
    hyb = case.flux_mode == W.FLUX_HYBRID
    weno = case.flux_mode != W.FLUX_CENTRAL
    conv = case.flux_mode != W.FLUX_WENO
    nprim = 6 + (2 if visc else 0) + (1 if weno else 0)        # rho u v w H p [T mu] [c]
    n_if = act["iface"] * N if hyb else (3 * N if weno else 0)
    n_sh = act["shock"] * N if hyb else (N if weno else 0)
    B, I = {}, {}
    # ghost shell only: the fused RHS kernel writes the primitives of the updated interior nodes (the one full pass
    # after streams_set_fields, 1 launch in 3 K, is not modelled): read the image, write the ghost w and primitives
    B["fill_prim"] = (Np - N) * (40 + 40 + 8 * nprim)
    I["fill_prim"] = (Np - N) * FP64_INST["fill_prim"]
    B["sensor"] = N * (24 + 8 + (1 if hyb else 0))             # read u v w, write div [mask]
    I["sensor"] = N * FP64_INST["sensor"]
    # shared-memory wavefronts of the sensor (the pipe that binds it): per node 2 L neighbours in x and in
    # y of three fields + three ring planes, 8-byte words: two 128-byte wavefronts per warp-wide load
    four = max(case.central_order // 2, (case.weno_order + 1) // 2 if weno else 0, case.visc_order // 2 if visc else 0) > 3
    Ls = 4 if four else case.central_order // 2
    SW = {"sensor": N * (3 * 4 * Ls + 3) * 2.0 / 32.0}
    B["flags"] = N * (1 + 1) + (n_if + n_sh) * 4               # read mask, write flags byte, append to the four work lists
    I["flags"] = 0
    # fused RHS + update: read 6 convective primitives [+ T mu div], read w, write w,
    # read R_prev (stages 2, 3), write R (stages 1, 2)
    # (+ hybrid / WENO: the flag byte of every node and the 5 net corrections of every node next to a flagged interface)
    # + the primitives of the updated node (a2 of the next stage), written to the other q buffer
    # (w: four fields read -- the old density comes with the primitives --, five written)
    per_point = (48 if conv else 0) + (24 if visc else 0) + 32 + 40 + (2.0 / 3.0) * 40 + (2.0 / 3.0) * 40 + 8 * nprim
    B["rhs_main"] = N * per_point + (N * 1 if hyb else 0) + n_sh * 40
    I["rhs_main"] = (N * FP64_INST["rhs_main_" + (("c" if conv else "") + ("v" if visc else "") or "0")]
                     + n_sh * FP64_INST["rhs_corr"] + N * (FP64_INST["prims"] + FP64_INST["fill_prim_dt"] / 3.0))
    # WENO: per flagged interface one new stencil node of 7 fields (runs of flagged interfaces share the
    # rest), a list entry, 5 flux values out
    B["weno"] = n_if * (56 + 4 + 40)                           # per timed group: the x, y and z launches of a stage
    I["weno"] = n_if * FP64_INST["weno_hybrid" if hyb else "weno_dense"]
    # net correction per listed node: list entry + flag byte, every interface value once, 5 values out
    B["corr_gather"] = (n_sh * 5 if hyb else 0) + n_if * 40 + n_sh * 40
    I["corr_gather"] = n_sh * FP64_INST["corr_gather"]
    B["dt"] = 0                                                # the rate is reduced inside fill_prim; this class is
    I["dt"] = 0                                                # the one-thread finalize (dt = CFL / rate)
    B["misc"] = 0
    I["misc"] = 0
    return B, I, per_point, SW


# ------------------------------------------------------------------------------------------------
# reference arm = the oracle on the host cores
# ------------------------------------------------------------------------------------------------
def oracle_throughput(case, budget_s: float, max_steps: int, kind: str = "omp"):
    """Times oracle RK3 steps of `case` (the build named by `kind`, as it stands) until budget_s is used or max_steps done."""
    from oracle.oracle import Oracle, load
    cores = int(load(kind).oracle_num_threads())
    ora = Oracle(case, kind=kind)
    done, t_used = 0, 0.0
    while done < max_steps and (done == 0 or t_used < budget_s):
        t0 = time.perf_counter()
        ora.step(1)
        t_used += time.perf_counter() - t0
        done += 1
    ora.close()
    return case.npoints * done / t_used, cores, done, t_used


def oracle_case_for(index: int):
    """The reference arm's bounded sample: the full workload when an oracle RK3 step takes seconds
    (configs 0-2), otherwise the same recipe on a grid cut to ~8 M points (CPU throughput per point does
    not depend on the grid size beyond cache effects)."""
    if index == 3:
        return W.boundary_layer(512, 128, 128, seed=3, nsteps=20), "same recipe on 512x128x128 (1/8 of the points)"
    if index == 5:
        return (W.isotropic_turbulence(nx=210, ny=125, nz=160, mach_t=0.6, k0=4.0, kmax=32, seed=5, nsteps=20,
                                       name="opt_iso_210x125x160"), "same recipe on 210x125x160 (1/8 of the points)")
    if index == 4:
        return (W.isotropic_turbulence(n=200, mach_t=0.8, k0=8.0, kmax=64, seed=4, nsteps=10, name="cfg4_iso_200"),
                "same recipe on 200^3 (1/33 of the points)")
    return make_case(index), "the full grid"


def serial_oracle_case_for(index: int):
    """The one-core sample: the same recipe on ~0.5 M points (an RK3 step of the serial oracle then takes seconds)."""
    if index == 0:
        return make_case(0), "the full grid"
    if index == 2:
        return W.channel(96, 72, 64, seed=2, nsteps=2), "same recipe on 96x72x64"
    if index == 3:
        return W.boundary_layer(192, 64, 48, seed=3, nsteps=2), "same recipe on 192x64x48"
    if index == 4:
        return (W.isotropic_turbulence(n=80, mach_t=0.8, k0=8.0, kmax=32, seed=4, nsteps=2, name="cfg4_iso_80"),
                "same recipe on 80^3")
    return (W.isotropic_turbulence(n=80, mach_t=0.6, k0=4.0, kmax=32, seed=1, nsteps=2, name="cfg1_iso_80"),
            "same recipe on 80^3")


def run_reference(args):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return 0
    case, what = oracle_case_for(args.config)
    from oracle.oracle import Oracle, load
    cores = int(load("omp").oracle_num_threads())
    ora = Oracle(case, kind="omp")
    for _ in range(args.warmup):
        ora.step(1)
    t0 = time.perf_counter()
    for _ in range(args.steps):
        ora.step(1)
    dt = time.perf_counter() - t0
    value = case.npoints * args.steps / dt
    sample = f"{args.steps} RK3 steps (3 RHS + update + dt each) of {what}, oracle OpenMP build"
    line = {
        "impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": 1e3 * dt / args.steps, "higher_is_better": True, "scaling": "weak",
        "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {"workload": WORKLOAD_TEXT[args.config], "grid": [case.nx, case.ny, case.nz],
                   "points": case.npoints, "sample": what, "device": "host CPU"},
        "cpu_baseline": {"value": value, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": sample},
        "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    print(json.dumps(line), flush=True)
    return 0


# ------------------------------------------------------------------------------------------------
# our arm: libstreams.so on the GPU through the C ABI
# ------------------------------------------------------------------------------------------------
def run_ours(args):
    import torch
    from paper_2304_05494_b200 import binding, build as kbuild, replicas

    rank, world, local = replicas.rank_info()
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device; libstreams has no CPU fallback (use --impl reference for the oracle)")
    torch.cuda.set_device(local)
    dist = None
    if world > 1:
        import torch.distributed as dist_mod
        dist = dist_mod
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))
    if rank == 0:
        kbuild.build()
    if dist is not None:
        dist.barrier()

    case = make_case(args.config, seed_offset=rank, cube=args.cube)
    # sweep knobs (not used by the default run): order family, flux mode, imposed activation
    m = args.order_family
    case = case.replace(central_order=2 * m, weno_order=2 * m - 1, visc_order=2 * m)
    if args.flux_mode:
        case = case.replace(flux_mode={"central": W.FLUX_CENTRAL, "weno": W.FLUX_WENO, "hybrid": W.FLUX_HYBRID}[args.flux_mode])
    N = case.npoints
    gpu = binding.Streams(case, device=f"cuda:{local}")
    dev = gpu.device
    if args.activation is not None:
        if case.flux_mode != W.FLUX_HYBRID:
            raise SystemExit("--activation needs hybrid mode")
        imposed = np.zeros((case.nz, case.ny, case.nx), dtype=np.uint8)
        imposed[: int(round(args.activation * case.nz))] = 1
        gpu.set_mask_override(imposed)
    state_bytes = 5 * N * 8


    rep = replicas.Replicas(dist, dev)          # barrier + max over ranks (tests/test_replicas_gloo.py)
    max_over_ranks = rep.max_over_ranks

    def sync_all():
        rep.barrier()
        torch.cuda.synchronize(dev)

    # Every timed region starts from the same state: the initial field advanced by `warmup` steps (the
    # workload is not stationary -- shocklets form and the WENO activation grows -- so regions that start
    # from different states are not comparable).
    gpu.step(args.warmup)
    w_start = torch.empty((5,) + gpu.shape, dtype=torch.float64, device=dev)
    gpu.get_fields(w_start)

    def timed_region(profile: bool):
        gpu.set_fields(w_start)
        for _ in range(3):                      # warm caches / clocks on the state itself (untimed)
            gpu.rhs()
        gpu.set_fields(w_start)                 # resets the activation totals too
        if profile:
            gpu.profile(True, max_records=10 * 3 * args.steps + 64)
        l0, g0 = gpu.kernel_launches(), gpu.graph_launches()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        sync_all()
        e0.record(gpu.stream)
        gpu.step(args.steps)
        e1.record(gpu.stream)
        sync_all()
        return max_over_ranks(e0.elapsed_time(e1)), (gpu.kernel_launches() - l0, gpu.graph_launches() - g0)

    # ---- device-resident throughput: inputs already in HBM, K steps in one streams_step call.  Two timed regions
    # of the same K steps from the same state: (1) the product path as a user runs it -> `value`; (2) the same with
    # the library's per-kernel CUDA event pairs on (streams_profile) -> the per-kernel roofline table; the event
    # pairs serialise the launches and cost 1-6 % (more on the tiny config 0), reported as `profiled`.
    timed_region(False)                         # one untimed pass of the whole region
    clocks = ClockSampler(local) if rank == 0 else None
    reps = []
    for _ in range(max(1, args.repeats)):       # best and median of >= 5 repeats from the same state
        ms_i, launches = timed_region(False)
        reps.append(ms_i)
    ms = float(np.median(reps))
    ms_prof, _ = timed_region(True)
    clk = clocks.stop() if clocks else None
    prof, dropped = gpu.get_profile()
    gpu.profile(False)
    flagged_sum, shock_sum, iface_sum, evals = gpu.get_activation_totals()
    act = {"flagged": flagged_sum / (evals * N) if evals else 0.0,
           "shock": shock_sum / (evals * N) if evals else 0.0,
           "iface": sum(iface_sum) / (evals * N) if evals else 0.0,
           "iface_xyz": [x / (evals * N) if evals else 0.0 for x in iface_sum]}
    value = world * N * args.steps / (ms * 1e-3)

    # ---- end to end through the C ABI with HOST buffers: every step copies the state host -> device,
    # advances it one RK3 step and copies it back; the state evolves through the host round trips
    h_a = torch.empty((5,) + gpu.shape, dtype=torch.float64).pin_memory()
    h_b = torch.empty((5,) + gpu.shape, dtype=torch.float64).pin_memory()
    gpu.set_fields(w_start)
    gpu.get_fields(h_a.numpy())
    n_e2e = max(3, min(args.steps, 20))
    for _ in range(2):
        gpu.set_fields(h_a.numpy()); gpu.step(1); gpu.get_fields(h_b.numpy())
    gpu.get_fields(h_b.numpy())
    sync_all()
    t0 = time.perf_counter()
    for _ in range(n_e2e):
        gpu.set_fields(h_a.numpy())       # host -> device (synchronous on return)
        gpu.step(1)
        gpu.get_fields(h_b.numpy())       # device -> host (synchronous on return)
        h_a, h_b = h_b, h_a
    torch.cuda.synchronize(dev)
    e2e_ms = max_over_ranks((time.perf_counter() - t0) * 1e3)
    e2e_value = world * N * n_e2e / (e2e_ms * 1e-3)
    assert np.isfinite(h_a.numpy()).all()

    if rank != 0:
        gpu.destroy()
        if dist is not None:
            dist.barrier()
            dist.destroy_process_group()
        return 0

    # ---- per-kernel roofline from the event pairs of the timed region
    peak, peak_src = load_peaks()
    sm_mhz = (clk or {}).get("sm_mhz") or 1965.0
    nominal_inst = N_SM * FP64_LANES_PER_SM * sm_mhz * 1e6     # fp64 thread-instructions / s at the clock under load
    # measured on this device through the C ABI (streams_measure_fp64): DFMA chains and DADD + DMUL chains
    fp64_meas = {"dfma_ginst_s": binding.measure_fp64(0, 5, gpu.stream), "dadd_dmul_ginst_s": binding.measure_fp64(1, 5, gpu.stream),
                 "nominal_ginst_s": nominal_inst / 1e9}
    peak_inst = fp64_meas["dfma_ginst_s"] * 1e9
    B, I, per_point, SW = work_model(case, act)
    peak_wave = N_SM * sm_mhz * 1e6                              # shared-memory wavefronts / s: one per SM and clock
    if args.order_family != 3:                  # the instruction counts were taken on the 6/5/6 instances
        I = {k: 0 for k in I}
    kernels = {}
    for name, (kms, cnt) in prof.items():
        if cnt == 0:
            continue
        t = kms / cnt * 1e-3
        gbs = B[name] / t / 1e9 if t > 0 else 0.0
        ginst = I[name] / t / 1e9 if t > 0 else 0.0
        t_hbm, t_alu = B[name] / (peak * 1e9), I[name] / peak_inst
        kernels[name] = {"launches": cnt, "avg_ms": t * 1e3, "share": kms / ms_prof, "alg_bytes": B[name], "gbs": gbs,
                         "frac_hbm": gbs / peak, "fp64_ginst_s": ginst, "frac_fp64": ginst * 1e9 / peak_inst,
                         "bound": "alu" if t_alu > t_hbm else "hbm", "frac": max(t_hbm, t_alu) / t if t > 0 else 0.0}
        if name in SW and t > 0:                # a kernel bound by the shared-memory data pipe (model count; ncu: profiles/)
            t_sm = SW[name] / peak_wave
            kernels[name].update({"smem_wavefronts": SW[name], "frac_smem": t_sm / t,
                                  "smem_peak": "148 SMs x 1 wavefront (128 B) / clk x %.0f MHz" % sm_mhz})
            if t_sm > max(t_hbm, t_alu):
                kernels[name].update({"bound": "smem", "frac": t_sm / t})
    dom = max(kernels, key=lambda k: kernels[k]["avg_ms"] * kernels[k]["launches"])
    kd = kernels[dom]
    if kd["bound"] == "hbm":
        roofline = {"kernel": dom, "bound": "hbm", "achieved": kd["gbs"], "peak": peak, "unit": "GB/s",
                    "frac": kd["frac_hbm"], "traffic": None, "peak_source": peak_src}
    else:   # fp64 pipe: 2 flop per instruction slot (DFMA), so 1 inst/s == 2 flop/s of the nominal peak
        roofline = {"kernel": dom, "bound": "alu", "achieved": 2 * kd["fp64_ginst_s"] / 1e3, "peak": 2 * peak_inst / 1e12,
                    "unit": "TFLOP/s", "frac": kd["frac_fp64"], "traffic": None,
                    "peak_source": "measured DFMA issue rate of this device (streams_measure_fp64) x 2 flop; nominal 148 SM x "
                                   "64 fp64 lanes x 2 x %.0f MHz = %.1f TFLOP/s; achieved counts every fp64 instruction as one "
                                   "FMA slot (DESIGN.md)" % (sm_mhz, 2 * nominal_inst / 1e12)}
    roofline.update({"alg_bytes_per_point_rhs_main": per_point, "kernels": kernels, "events_dropped": dropped,
                     "hbm_peak_gbs": peak, "hbm_peak_source": peak_src, "fp64_peak": fp64_meas})
    traffic_file = os.path.join(ROOT, "profiles", "traffic.json")
    if os.path.exists(traffic_file):           # dram bytes per launch from the committed ncu --set full capture
        with open(traffic_file) as f:
            tr = json.load(f)
        key = f"cfg{args.config}:{dom}"
        if key in tr:
            # the capture is a separate run under ncu: say at which activation (flagged interfaces per node) and step
            # counts it was taken, and do not quote its bytes beside a timed region that sat elsewhere (the traffic of
            # every kernel but the sensor grows with the activation)
            cap_act, here = tr[key].get("iface_per_node"), act["iface"]
            comparable = (not case_is_hybrid(case)) or (cap_act is not None and abs(cap_act - here) <= 0.2 * max(here, 1e-12))
            roofline["traffic"] = tr[key]["dram_bytes_per_launch"] if comparable else None
            roofline["traffic_source"] = tr[key].get("source")
            roofline["traffic_capture"] = {"iface_per_node": cap_act, "command": tr[key].get("command"),
                                           "iface_per_node_timed_region": here, "comparable": comparable,
                                           "dram_bytes_per_launch": tr[key]["dram_bytes_per_launch"]}

    # ---- the oracle on this box's host cores (bounded sample, rank 0, N = 1 only)
    cpu = None
    if world == 1 and not args.no_cpu_baseline:
        ocase, what = oracle_case_for(args.config)
        v, cores, done, used = oracle_throughput(ocase, budget_s=12.0, max_steps=args.steps)
        cpu = {"value": v, "unit": UNIT, "cores": cores, "kind": "oracle",
               "sample": f"{done} RK3 steps of {what} ({used:.1f} s), oracle OpenMP build as it stands"}
        # the serial build on one core (SURVEY 8(d) "the reported CPU baseline"; PAPER:357-359 quotes per-core context):
        # a smaller sample of the same recipe so that one RK3 step takes seconds
        scase, swhat = serial_oracle_case_for(args.config)
        v1, c1, d1, u1 = oracle_throughput(scase, budget_s=10.0, max_steps=2, kind="serial")
        cpu["serial"] = {"value": v1, "unit": UNIT, "cores": c1, "kind": "oracle",
                         "sample": f"{d1} RK3 steps of {swhat} ({u1:.1f} s), oracle serial build as it stands"}

    line = {
        "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
        "ms_per_step": ms / args.steps, "repeats": {"n": len(reps), "median_ms_per_step": ms / args.steps,
                                                    "best_ms_per_step": min(reps) / args.steps,
                                                    "worst_ms_per_step": max(reps) / args.steps,
                                                    "best_value": world * N * args.steps / (min(reps) * 1e-3),
                                                    "note": "`value` is the median region"},
        "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
        "dtype": "f64", "data": "synthetic",
        "config": {"workload": WORKLOAD_TEXT[args.config], "grid": [case.nx, case.ny, case.nz], "points": N,
                   "orders": "central %d / WENO %d / viscous %d" % (case.central_order, case.weno_order, case.visc_order),
                   "flux_mode": {W.FLUX_CENTRAL: "central", W.FLUX_WENO: "weno", W.FLUX_HYBRID: "hybrid"}[case.flux_mode],
                   "imposed_activation": args.activation, "parallelism": "1 GPU" if world == 1 else
                   f"{world} independent replicas (no data-path collective)",
                   "l2": "inputs larger than L2 (workspace %.2f GB vs 126 MB)" % (gpu.workspace_bytes / 1e9)
                   if gpu.workspace_bytes > 4 * 126e6 else "workspace %.1f MB is L2-resident; latency point, not a roofline point"
                   % (gpu.workspace_bytes / 1e6),
                   "weno_activation": act},
        "clocks": clk,
        "e2e": {"value": e2e_value, "unit": UNIT, "h2d_bytes_per_step": state_bytes, "d2h_bytes_per_step": state_bytes,
                "steps": n_e2e, "ms_per_step": e2e_ms / n_e2e},
        "gpu_launches": launches[0],
        "graph_launches": launches[1],
        "library": os.environ.get("STREAMS_LIB") or "paper_2304_05494_b200/lib/libstreams.so",
        "roofline": roofline,
        "cpu_baseline": cpu,
        "point_stages_per_s": 3 * value,
        "profiled": {"value": world * N * args.steps / (ms_prof * 1e-3), "ms_per_step": ms_prof / args.steps,
                     "note": "the same K steps with per-kernel event pairs on; roofline.kernels (avg_ms, share) come from this region"},
        "paper_context": "A100 1.06e8 (central) / 7.05e7 (WENO) point-steps/s on 420x250x320, PAPER:398-404 (other hardware)",
    }
    print(json.dumps(line), flush=True)
    gpu.destroy()
    if dist is not None:
        dist.barrier()
        dist.destroy_process_group()
    return 0


# ------------------------------------------------------------------------------------------------
# sharded arm: ONE problem cut into z slabs, halo exchange per phase (strong scaling)
# ------------------------------------------------------------------------------------------------
def run_sharded(args):
    """`--sharded`: the config's grid is cut into z slabs, one per rank (torchrun, NCCL point-to-point between
    neighbours) or `--slabs S` slabs inside this process when there is one GPU (the copies are then device copies on one
    stream; this measures what the phase structure and the exchange cost, not a speed-up).  value = points of the WHOLE
    grid x K / max-over-ranks device time."""
    import torch
    from paper_2304_05494_b200 import build as kbuild, replicas, sharded

    rank, world, local = replicas.rank_info()
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device; libstreams has no CPU fallback")
    torch.cuda.set_device(local)
    dist = None
    if world > 1:
        import torch.distributed as dist_mod
        dist = dist_mod
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))
    if rank == 0:
        kbuild.build()
    if dist is not None:
        dist.barrier()
    case = make_case(args.config)                   # every rank builds the same field and keeps its slab
    nslabs = world if world > 1 else max(1, args.slabs)
    ranks = [rank] if world > 1 else list(range(nslabs))
    sh = sharded.ShardedStreams(case, nslabs, ranks, device=f"cuda:{local}", dist=dist)
    rep = replicas.Replicas(dist, sh.device)
    N = case.npoints
    sh.step(args.warmup)
    snap = sh.snapshot()                            # every region starts from the same state (the activation grows with time)
    clocks = ClockSampler(local) if rank == 0 else None
    reps = []
    for _ in range(max(1, args.repeats)):
        sh.restore(snap)
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        rep.barrier(); torch.cuda.synchronize(sh.device)
        e0.record(sh.stream)
        sh.step(args.steps)
        e1.record(sh.stream)
        rep.barrier(); torch.cuda.synchronize(sh.device)
        reps.append(rep.max_over_ranks(e0.elapsed_time(e1)))
    clk = clocks.stop() if clocks else None
    ms = float(np.median(reps))
    launches = sh.kernel_launches()
    halo_bytes = sh.halo_bytes_per_stage()          # from the slab sizes streams_halo_slabs reports (any ghost width)
    w = sh.get_fields()
    ok = bool(np.isfinite(w).all())
    sh.destroy()
    if rank == 0:
        ranges = sharded.slab_ranges(case.nz, nslabs)
        line = {
            "metric": METRIC, "value": N * args.steps / (ms * 1e-3), "unit": UNIT, "n_gpus": world, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": ms / args.steps,
            "repeats": {"n": len(reps), "best_ms_per_step": min(reps) / args.steps, "median_ms_per_step": ms / args.steps},
            "higher_is_better": True, "scaling": "strong", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": WORKLOAD_TEXT[args.config], "grid": [case.nx, case.ny, case.nz], "points": N,
                       "parallelism": (f"{nslabs} z slabs, one per GPU, halo exchange by NCCL send / receive" if world > 1 else
                                       f"{nslabs} z slabs in one process on one GPU (exchange = device copies)"),
                       "slab_planes": [b - a for a, b in ranges], "halo_bytes_sent_per_slab_per_stage": halo_bytes,
                       "l2": "inputs larger than L2" if N * 400 > 4 * 126e6 else "L2-resident"},
            "clocks": clk, "gpu_launches": launches, "state_finite": ok, "roofline": None, "cpu_baseline": None,
            "e2e": None,
        }
        print(json.dumps(line), flush=True)
    if dist is not None:
        dist.barrier()
        dist.destroy_process_group()
    return 0


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=None, help="timed RK3 steps per region (default: the config's own count)")
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--config", type=int, default=4,
                    help="index into BASELINE.json configs (default 4: the largest single-GPU configuration)")
    ap.add_argument("--cube", type=int, default=256, help="--config 6 (size sweep): N of the N^3 periodic box")
    ap.add_argument("--repeats", type=int, default=5, help="timed regions from the same state; value = median")
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--order-family", type=int, default=3, choices=[1, 2, 3, 4],
                    help="m: central order 2m / WENO order 2m-1 / viscous order 2m (default 3 = 6/5/6)")
    ap.add_argument("--flux-mode", default=None, choices=["central", "weno", "hybrid"], help="override the config's flux mode")
    ap.add_argument("--sharded", action="store_true",
                    help="cut the grid into z slabs (one per rank under torchrun, --slabs in one process otherwise) "
                         "and exchange halo planes every phase: strong scaling instead of independent replicas")
    ap.add_argument("--slabs", type=int, default=2, help="--sharded on one GPU: number of slabs in this process")
    ap.add_argument("--activation", type=float, default=None,
                    help="hybrid mode: impose the node mask on this fraction of the z planes (PAPER:497-501 sweep)")
    args = ap.parse_args()
    if args.steps is None:
        args.steps = {0: 10, 1: 50, 2: 50, 3: 20, 4: 10, 5: 20}.get(args.config, 20) if args.impl == "ours" else 3
    if args.warmup < 3 and args.impl == "ours":
        args.warmup = 3
    if args.impl == "reference":
        return run_reference(args)
    if args.sharded:
        return run_sharded(args)
    return run_ours(args)


if __name__ == "__main__":
    sys.exit(main())
