#!/usr/bin/env python
"""bench.py -- MTP energy+force atom-evaluations/s on one B200 (or N replicas, weak scaling).

A "step" is one pass of the whole hot path (rows a1-a8, a10 of SURVEY.md 8(a)) over one BASELINE.json
workload; the default is configs[3], the one the metric is quoted on: 1,048,576 atoms, 3 species, FCC 64^3,
level 16, fp64, chunked evaluation.  `value` is device-resident throughput (CUDA events), `e2e` the same metric
through mtp_compute_host_pos with pinned HOST buffers (H2D + D2H inside the timed region; `e2e_host_list`: through
mtp_compute_host, the caller's list copied as well), `md` the device MD loop in atom-timesteps/s.  `--impl reference`
times the CPU oracle (oracle/, as it stands) on a bounded sample, on all host cores; it does not load the
CUDA library.

  python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference]
                  [--config I] [--cells C] [--grade]        (the last three: profiling aids)
"""
from __future__ import annotations

import argparse
import json
import multiprocessing
import os
import socket
import subprocess
import sys
import tempfile
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

LEVELS = [10, 16, 20, 16, 24]
HEADLINE = 3                         # 0-based index of the configuration BASELINE.json's metric is quoted on
UNIT = "atom-evals/s"
MD_DT = 1e-10                        # ps, upper bound of the MD leg's time step (it is reduced further where the forces ask for it)


def metric_name(config, w):
    """BASELINE.json's metric string for the configuration it is quoted on; the other configs say what they are."""
    if config == HEADLINE and w.n_atoms == 1048576:
        return "MTP energy+force atom-evals/s at ~1M atoms lev16 fp64"
    return "MTP energy+force atom-evals/s at %d atoms lev%d fp64" % (w.n_atoms, w.lev_max)


def flops_per_step(cost, n_pairs, n_atoms):
    """Algorithmic flops of one step per kernel class (FMA = 2, each quantity once; formulas: DESIGN.md section 6,
    numbers from mtp_cost_model) for the pairs and atoms this rank evaluates."""
    return {"moments": cost["flop_per_pair_k1"] * n_pairs, "pairgrad": cost["flop_per_pair_k3"] * n_pairs,
            "tree": cost["flop_per_atom_tree"] * n_atoms}


class ClockSampler:
    """nvidia-smi clocks / throttle reasons during the timed region (B200_PROFILING.md)."""

    Q = ("index,clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.active,"
         "clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
         "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, gpu_index):
        self.path = tempfile.mktemp(prefix="mtp_clocks_", suffix=".csv")
        self.gpu = gpu_index
        self.proc = None

    def start(self):
        try:
            self.f = open(self.path, "w")
            self.proc = subprocess.Popen(["nvidia-smi", "-i", str(self.gpu), "--query-gpu=" + self.Q,
                                          "--format=csv,noheader,nounits", "-lms", "50"],
                                         stdout=self.f, stderr=subprocess.DEVNULL)
        except Exception:
            self.proc = None

    def stop(self):
        out = dict(sm_mhz=None, sm_max_mhz=None, reasons=[])
        if self.proc is None:
            return out
        time.sleep(0.15)
        self.proc.terminate()
        try:
            self.proc.wait(timeout=5)
        except Exception:
            self.proc.kill()
        self.f.close()
        sm, mx, reasons = [], [], set()
        for line in open(self.path):
            p = [x.strip() for x in line.split(",")]
            if len(p) < 9:
                continue
            try:
                sm.append(float(p[1])); mx.append(float(p[2]))
            except ValueError:
                continue
            for name, v in zip(("hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"), p[5:9]):
                if v.lower().startswith("active"):
                    reasons.add(name)
        os.unlink(self.path)
        if sm:
            out = dict(sm_mhz=float(np.median(sm)), sm_max_mhz=float(max(mx)), reasons=sorted(reasons),
                       samples=len(sm))
        return out


def max_over_ranks(x, dist, device):
    """Time of the slowest rank (the contract's max-over-ranks); identity for a single process."""
    if dist is None:
        return float(x)
    import torch
    t = torch.tensor([float(x)], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def whole_job_rate(n_atoms_per_rank, steps, seconds_local, world, dist, device):
    """Weak scaling over replicas: every rank evaluates its own n_atoms_per_rank atoms per step;
    value = atoms all ranks processed / time of the slowest rank."""
    return world * n_atoms_per_rank * steps / max_over_ranks(seconds_local, dist, device)


def build_workload(config, cells, n_basis, seed_shift=0):
    """The seeded synthetic workload (workloads/ holds no method arithmetic).  n_basis comes from the caller's own
    basis enumeration: the CUDA library's for our arm, the oracle's for the reference arm."""
    from workloads import make_workload, CONFIGS
    from workloads.lattice import BASE_SEED
    w = make_workload(config, n_basis, cells=cells, with_ainv=None, seed=BASE_SEED + config + 1000 * seed_shift)
    return w, CONFIGS[config]


def config_dict(w, cfg, world, sharded=False):
    """What the workload is -- the same dictionary in both arms."""
    return {"workload": cfg["name"], "n_atoms": w.n_atoms, "nnz": w.nnz, "lev_max": w.lev_max, "n_species": w.n_species,
            "n_basis": int(w.xi.shape[0]),
            "l2": ("inputs larger than L2 (neighbour list %.0f MB + per-pair scratch), no flush" % (w.nnz * 11 / 1e6)) if w.nnz * 43 > 126e6
                  else "inputs and scratch fit in the 126 MB L2 and are not flushed: L2-warm steady state, as between the steps of an MD run",
            "parallelism": ("atom ranges x%d, all-reduce of F" if sharded else "replicas x%d") % world}


# ---------------------------------------------------------------- the oracle, timed on the host cores
_ORACLE = {}


def _oracle_worker(rng):
    from oracle import mtp as omtp
    w, pot = _ORACLE["w"], _ORACLE["pot"]
    omtp.evaluate(pot, w.pos, w.types, w.box, w.off, w.idx, w.shift, atoms=range(rng[0], rng[1]), want_grad=True)
    return rng[1] - rng[0]


def host_cores():
    try:
        return max(1, len(os.sched_getaffinity(0)))
    except Exception:
        return max(1, os.cpu_count() or 1)


class OraclePool:
    """The oracle as it stands (oracle/mtp.py evaluate: E_i, d_ij, force scatter per atom), one single-threaded
    process per host core over contiguous atom ranges of the same workload.  Forked before CUDA is touched."""

    def __init__(self, w, cores):
        from oracle import mtp as omtp
        try:
            from threadpoolctl import threadpool_limits
            threadpool_limits(limits=1)
        except Exception:
            pass
        _ORACLE["w"] = w
        _ORACLE["pot"] = omtp.Potential(w.lev_max, w.n_mu, w.n_beta, w.r_min, w.r_cut, w.c, w.xi0, w.xi)
        self.cores = cores
        self.pool = multiprocessing.get_context("fork").Pool(cores) if cores > 1 else None

    def rate(self, w, atoms_per_core):
        n = min(w.n_atoms, atoms_per_core * self.cores)
        per = (n + self.cores - 1) // self.cores
        ranges = [(lo, min(n, lo + per)) for lo in range(0, n, per)]
        t0 = time.perf_counter()
        done = sum(self.pool.map(_oracle_worker, ranges)) if self.pool else sum(_oracle_worker(r) for r in ranges)
        dt = time.perf_counter() - t0
        return done / dt, dt, done

    def close(self):
        if self.pool:
            self.pool.close()
            self.pool.join()


def run_reference(args):
    """--impl reference: the oracle timed on the host cores; each step is a bounded sample.  Loads nothing of the
    CUDA library: n_basis is the oracle's own enumeration."""
    if int(os.environ.get("RANK", "0")) != 0:
        return
    from oracle import basis as obasis
    n_basis = len(obasis.basis_functions(LEVELS[args.config]))
    w, cfg = build_workload(args.config, args.cells, n_basis)
    cores = host_cores()
    pool = OraclePool(w, cores)
    per_core = args.ref_atoms or 1024           # x (steps + warmup): the whole run stays within a few minutes
    for _ in range(args.warmup):
        pool.rate(w, max(64, per_core // 8))
    t = 0.0
    n = 0
    for _ in range(args.steps):
        _, dt, k = pool.rate(w, per_core)
        t += dt
        n += k
    pool.close()
    value = n / t
    sample = "first %d atoms of the workload per step (E_i, d_ij, force scatter), %d processes" % (n // max(args.steps, 1), cores)
    line = {
        "impl": "reference", "metric": metric_name(args.config, w), "value": value, "unit": UNIT, "n_gpus": args.gpus,
        "steps": args.steps, "warmup": args.warmup, "ms_per_step": 1e3 * t / max(args.steps, 1),
        "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": config_dict(w, cfg, 1),
        "cpu_baseline": {"value": value, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": sample},
        "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    print(json.dumps(line), flush=True)


def graph_replay(torch, pot, graph, calls=100):
    """small configurations additionally through the library's own CUDA graph of the call
    (mtp_graph_capture / mtp_graph_launch: one launch per evaluation, the per-kernel launch overhead gone); ms per call."""
    for _ in range(3):
        graph.launch()
    torch.cuda.synchronize()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record()
    for _ in range(calls):
        graph.launch()
    e1.record()
    torch.cuda.synchronize()
    return e0.elapsed_time(e1) / calls


def load_traffic(workload, kernel):
    """dram bytes per launch of `kernel` from the committed ncu capture of THIS workload (profiles/traffic.json,
    keyed by workload name), else None: the number is not measurable without ncu."""
    tpath = os.path.join(ROOT, "profiles", "traffic.json")
    try:
        return json.load(open(tpath)).get(workload, {}).get(kernel)
    except Exception:
        return None


def run_ours(args):
    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))

    import paper_2510_00193_b200 as lib           # raises if libmtp_b200.so is missing: there is no fallback
    table = lib.Table(LEVELS[args.config])
    # replicas (default, weak scaling): every rank its own seeded system; --sharded (strong scaling): one system, the
    # atoms cut into contiguous ranges, one all-reduce of the partial forces per step (paper_2510_00193_b200/sharded.py)
    w, cfg = build_workload(args.config, args.cells, table.n_basis, seed_shift=0 if args.sharded else rank)

    # ---- CPU baseline first (processes are forked before this process touches CUDA): the oracle on a bounded
    # sample of the same workload, all host cores
    cpu = None
    if world == 1 and not args.no_cpu_baseline:
        cores = host_cores()
        pool = OraclePool(w, cores)
        rate, dt, k = pool.rate(w, args.ref_atoms or 8192)
        pool.close()
        cpu = {"value": rate, "unit": UNIT, "cores": cores, "kind": "oracle",
               "sample": "first %d atoms of the workload (E_i, d_ij, force scatter), %d processes, %.1f s" % (k, cores, dt)}

    import torch
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: there is no CPU fallback")
    torch.cuda.set_device(local)
    dev = torch.device("cuda", local)
    dist = None
    if world > 1:
        import torch.distributed as dist_
        dist = dist_
        dist.init_process_group("nccl", device_id=dev)

    pot = lib.Potential(table, w.n_species, w.n_beta, w.r_min, w.r_cut, w.c, w.xi0, w.xi)
    if args.chunk >= 0:
        pot.set_option(lib.OPT_CHUNK_ATOMS, args.chunk)
    if args.force_mode >= 0:
        pot.set_option(lib.OPT_FORCE_MODE, args.force_mode)
    pot.set_option(lib.OPT_PROFILE, 1)
    t = lambda a, dt: torch.as_tensor(np.ascontiguousarray(a), dtype=dt).to(dev)
    pos, types, off, idx = t(w.pos, torch.float64), t(w.types, torch.int32), t(w.off, torch.int64), t(w.idx, torch.int32)
    shift, rev = t(w.shift, torch.int8), t(w.rev, torch.int32)
    Ainv = t(w.Ainv, torch.float64) if (args.grade and w.Ainv is not None) else None

    if args.sharded:
        from paper_2510_00193_b200 import sharded
        lo, hi = sharded.balanced_row_range(w.off, rank, world)
        off_w, idx_w, shift_w = (t(a, dt) for a, dt in zip(sharded.window_list(w.off, w.idx, w.shift, lo, hi),
                                                           (torch.int64, torch.int32, torch.int8)))

    def step(out=None):
        if args.sharded:
            o = pot.compute_rows(pos, types, w.box, lo, hi, off_w, idx_w, shift_w, out=out)
            if dist is not None:
                sharded.all_reduce_sum(dist, o["F"], o["E"], o["virial"])
            return o
        o = pot.compute(pos, types, w.box, off, idx, shift, rev, out=out)
        if Ainv is not None:
            pot.grade(pos, types, w.box, off, idx, Ainv, shift, mode=2)
        return o

    def barrier():
        if dist is not None:
            dist.barrier()
        torch.cuda.synchronize()

    out = None
    for _ in range(max(args.warmup, 0)):
        out = step(out)
    torch.cuda.synchronize()
    pot.profile_read()
    sampler = ClockSampler(local)
    barrier()
    sampler.start()
    n0 = lib.launch_count()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record()
    for _ in range(args.steps):
        out = step(out)
    e1.record()
    barrier()
    clocks = sampler.stop()
    launches = lib.launch_count() - n0
    ms = e0.elapsed_time(e1)
    prof = pot.profile_read()
    ms = max_over_ranks(ms, dist, dev)
    # replicas: every rank evaluated its own n_atoms; sharded: the ranks evaluated one system together
    value = whole_job_rate(w.n_atoms, args.steps, ms * 1e-3, 1 if args.sharded else world, None, dev)

    # ---- small systems: the same call replayed from a CUDA graph (launch overhead removed)
    graph = None
    if w.n_atoms <= 16384 and Ainv is None and world == 1 and not args.sharded:
        try:
            cg, gout = pot.graph(pos, types, w.box, off, idx, shift, rev)
            gms = graph_replay(torch, pot, cg)
            assert torch.equal(gout["F"], out["F"]), "graph launch differs from mtp_compute"
            cg.close()
            graph = {"calls": 100, "ms_per_call": gms, "value": w.n_atoms / (gms * 1e-3), "unit": UNIT,
                     "entry": "mtp_graph_capture / mtp_graph_launch"}
        except Exception as exc:      # an auxiliary leg must not take the headline line with it
            graph = {"error": "%s: %s" % (type(exc).__name__, exc)}

    # ---- end to end through the host-buffer entry points (pinned inputs, results read back).  `e2e`: what an MD host
    # code sends every step -- positions and types -- with the list built on the device (mtp_compute_host_pos);
    # `e2e_host_list`: the caller's own list copied too (mtp_compute_host; "the GPU runs use the host
    # code's list")
    pin = lambda a: torch.from_numpy(np.ascontiguousarray(a)).pin_memory().numpy()
    hp = dict(pos=pin(w.pos), types=pin(w.types), off=pin(w.off), idx=pin(w.idx), shift=pin(w.shift), rev=pin(w.rev))
    hout = dict(E=pin(np.zeros(1)), Ei=pin(np.zeros(w.n_atoms)), F=pin(np.zeros((w.n_atoms, 3))), virial=pin(np.zeros(6)))
    e2e_steps = max(1, min(args.steps, 10))

    def timed_host(call):
        call()
        barrier()
        t0 = time.perf_counter()
        for _ in range(e2e_steps):
            call()
        torch.cuda.synchronize()
        return whole_job_rate(w.n_atoms, e2e_steps, time.perf_counter() - t0, world, dist, dev)


    # (the host entry points and the MD loop evaluate a whole system per rank: these legs are replicas in either mode)
    e2e_list_value = timed_host(lambda: pot.compute_host(hp["pos"], hp["types"], w.box, hp["off"], hp["idx"], hp["shift"], hp["rev"], out=hout))
    h2d_list = sum(hp[k].nbytes for k in hp)
    e2e_value = timed_host(lambda: pot.compute_host_pos(hp["pos"], hp["types"], w.box, out=hout))
    assert hout["nnz"] == w.nnz, "device list differs from the workload's"
    h2d = hp["pos"].nbytes + hp["types"].nbytes
    d2h = sum(hout[k].nbytes for k in ("E", "Ei", "F", "virial"))
    pot.profile_read()

    # ---- MD loop on the device: velocity-Verlet steps with the list rebuilt every 10 steps at a
    # 1 A skin, atom-timesteps/s (the paper's unit, list builds included).  The seeded random
    # coefficients make a stiff potential, hence the tiny time step MD_DT: the work per step does not depend on it.
    md = None
    if not args.no_md and Ainv is None:
        try:
            md_steps = max(10, min(args.steps, 50))
            cap = int(w.nnz * 1.9) + 1024                       # (6 / 5)^3 = 1.73 x the pairs at R_cut
            mpos, mvel = pos.clone(), torch.zeros_like(pos)
            mass = np.full(w.n_species, 55.845)
            # the atoms must stay put over the 10 + md_steps steps (forces reach 1e8 eV/A at level 16 and far more at level
            # 24 with the seeded coefficients): a step such that the largest acceleration moves an atom by < 1e-3 A in total
            a_max = 9648.533 * float(out["F"].abs().max().item()) / mass[0]
            md_dt = min(MD_DT, (2e-3 / max(a_max, 1e-300)) ** 0.5 / (10 + md_steps))
            pot.set_option(lib.OPT_PROFILE, 0)
            pot.md_run(mpos, mvel, types, w.box, mass, md_dt, 10, 10, 1.0, cap)
            barrier()
            n1 = lib.launch_count()
            m0, m1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            m0.record()
            mo = pot.md_run(mpos, mvel, types, w.box, mass, md_dt, md_steps, 10, 1.0, cap)
            m1.record()
            barrier()
            md_ms = max_over_ranks(m0.elapsed_time(m1), dist, dev)
            info = [int(x) for x in mo["info"].cpu()]
            assert info[0] <= cap and info[1] == 0, "MD list overflow"
            md = {"value": world * w.n_atoms * md_steps / (md_ms * 1e-3), "unit": "atom-timesteps/s", "steps": md_steps,
                  "ms_per_step": md_ms / md_steps, "rebuild_every": 10, "skin": 1.0, "dt_ps": md_dt, "list_pairs": info[0],
                  "gpu_launches": int(lib.launch_count() - n1)}
            pot.set_option(lib.OPT_PROFILE, 1)
            del mpos, mvel, mo
        except Exception as exc:      # an auxiliary leg must not take the headline line with it
            md = {"error": "%s: %s" % (type(exc).__name__, exc)}
            pot.set_option(lib.OPT_PROFILE, 1)

    if rank != 0:
        if dist is not None:
            dist.destroy_process_group()
        return

    # ---- roofline of the dominant kernel (fp64 ALU bound)
    per_step = flops_per_step(pot.cost_model(), int(w.off[hi] - w.off[lo]), hi - lo) if args.sharded else \
        flops_per_step(pot.cost_model(), w.nnz, w.n_atoms)
    timed = {k: prof[k] for k in ("moments", "tree", "pairgrad")}
    if Ainv is not None:                                   # --grade: K5's GEMM, 2 n_basis^2 flop per atom (fp64 mma.sync: the same peak)
        per_step["grade"] = 2.0 * float(table.n_basis) ** 2 * (hi - lo if args.sharded else w.n_atoms)
        timed["grade"] = prof["grade"]
    dom = max(timed, key=lambda k: timed[k][0])
    dom_ms, dom_n = timed[dom]
    sms = torch.cuda.get_device_properties(dev).multi_processor_count
    sm_ghz = (clocks.get("sm_max_mhz") or 1965.0) / 1e3
    peak_tf = sms * 64 * 2 * sm_ghz * 1e9 / 1e12       # 64 fp64 FMA / clk / SM at clocks.max.sm
    achieved_tf = per_step[dom] * args.steps / (dom_ms * 1e-3) / 1e12 if dom_ms > 0 else 0.0
    step_tf = sum(per_step.values()) * args.steps / (ms * 1e-3) / 1e12
    # measured DFMA throughput of this box (own microbenchmark, reported beside the derived peak)
    sink = torch.zeros(8, dtype=torch.float64, device=dev)
    lib.peak_dfma(2000, sink)
    torch.cuda.synchronize()
    a0, a1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    a0.record()
    pk = lib.peak_dfma(20000, sink)
    a1.record()
    torch.cuda.synchronize()
    measured_tf = pk / (a0.elapsed_time(a1) * 1e-3) / 1e12
    ws_bytes = pot.workspace_bytes(w.n_atoms, w.nnz)

    line = {
        "metric": metric_name(args.config, w), "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": ms / args.steps, "higher_is_better": True,
        "scaling": "strong" if args.sharded else "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": config_dict(w, cfg, world, args.sharded),
        "run": {"chunk_atoms": pot.get_option(lib.OPT_CHUNK_ATOMS), "force_mode": pot.get_option(lib.OPT_FORCE_MODE),
                "grade": bool(Ainv is not None), "tree_kernels": pot.get_option(lib.INFO_TREE_KERNELS),
                "tree_programs": pot.get_option(lib.INFO_TREE_PROGRAMS), "tree_note": pot.last_error(),
                "workspace_bytes": int(ws_bytes)},
        "clocks": clocks,
        "e2e": {"value": e2e_value, "unit": UNIT, "h2d_bytes_per_step": int(h2d), "d2h_bytes_per_step": int(d2h),
                "steps": e2e_steps, "entry": "mtp_compute_host_pos (positions in, list built on the device)"},
        "e2e_host_list": {"value": e2e_list_value, "unit": UNIT, "h2d_bytes_per_step": int(h2d_list),
                          "d2h_bytes_per_step": int(d2h), "steps": e2e_steps, "entry": "mtp_compute_host (caller's list copied)"},
        "gpu_launches": int(launches),
        "roofline": {"bound": "alu", "kernel": dom, "achieved": achieved_tf, "peak": peak_tf, "unit": "TFLOP/s",
                     "frac": achieved_tf / peak_tf, "traffic": load_traffic(cfg["name"], dom),
                     "peak_source": "derived: %d SMs x 64 fp64 FMA/clk x 2 x %.3f GHz (clocks.max.sm); MEASURED_PEAKS.json has no fp64 entry; "
                                    "own DFMA microbenchmark in this run %.1f TF/s" % (sms, sm_ghz, measured_tf),
                     "flops_per_launch": per_step[dom] / max(dom_n / args.steps, 1), "launches": dom_n,
                     "avg_launch_ms": dom_ms / max(dom_n, 1),
                     "step_achieved": step_tf, "step_frac": step_tf / peak_tf,
                     "kernel_ms_per_step": {k: v[0] / args.steps for k, v in prof.items()}},
        "cpu_baseline": cpu,
    }
    if graph is not None:
        line["graph_replay"] = graph
    if md is not None:
        line["md"] = md
    print(json.dumps(line), flush=True)
    if dist is not None:
        dist.destroy_process_group()


def spawn_ranks(args):
    """`python bench.py --gpus N` outside torchrun: re-run this script as N ranks of one node."""
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        port = s.getsockname()[1]
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node", str(args.gpus),
           "--master-addr", "127.0.0.1", "--master-port", str(port), os.path.abspath(__file__)] + sys.argv[1:]
    raise SystemExit(subprocess.call(cmd))


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=50)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--config", type=int, default=HEADLINE, help="0-based index into BASELINE.json configs")
    ap.add_argument("--cells", type=int, default=None, help="override the lattice repeat (scaled-down instance)")
    ap.add_argument("--chunk", type=int, default=-1)
    ap.add_argument("--force-mode", type=int, default=-1)
    ap.add_argument("--grade", action="store_true", help="also run mtp_grade each step (config 4)")
    ap.add_argument("--ref-atoms", type=int, default=None,
                    help="atoms per core of an oracle sample (default: 8192 for cpu_baseline, 1024 per step for --impl reference)")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-md", action="store_true", help="skip the MD-loop leg")
    ap.add_argument("--sharded", action="store_true",
                    help="N > 1: one system cut into atom ranges with an all-reduce of F per step (strong scaling) instead of replicas")
    args = ap.parse_args()
    if args.impl == "reference":
        run_reference(args)
    elif args.gpus > 1 and "WORLD_SIZE" not in os.environ:
        spawn_ranks(args)
    else:
        run_ours(args)


if __name__ == "__main__":
    main()
