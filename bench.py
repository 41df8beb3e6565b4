#!/usr/bin/env python
"""bench.py -- throughput of the LEDDS hot path on B200.

A "step" is one pass of the whole hot path: one coupled LBM-DEM step of
BASELINE.json configs[3] (256^3 D3Q19 BGK lattice, periodic x/y, moving z walls, 20 000 spheres of
radius 4 placed by seeded RSA, PSM coupling, n_sub = 1).  The headline value is MLUPS from the
total time per step including DEM and coupling (the paper's own definition).
Sub-benchmarks are reported in the same JSON line under "sub": configs[1] LBM-only MLUPS (BGK and TRT),
configs[0] and configs[2] (latency-bound; plain and from a CUDA graph), configs[4] DEM-only
particle-updates/s with GB/s per kernel, configs[3] with TRT + subdivision solid fraction, and the paper's
own 500x200x800 performance workload at four solid fractions.  Multi-GPU (N > 1, torchrun) = independent replicas, no collective
on the data path ("replicas only").

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference] [--workload cfg4|small] [--no-sub]
"""
import argparse
import json
import os
import subprocess
import sys
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

METRIC = "D3Q19 MLUPS of the coupled LBM-DEM step (total time per step incl. DEM and coupling)"


NOMINAL_HBM_GBS = 8000.0        # the "~8 TB/s" of north_star (HGX figure 7.7 TB/s); context next to the measured copy rate


def peaks():
    try:
        return json.load(open(os.path.join(ROOT, "MEASURED_PEAKS.json")))["hbm_gbs"], "measured (MEASURED_PEAKS.json)"
    except Exception:
        return 6650.0, "fallback (B200_PROFILING.md)"


def fracs(gbs, peak):
    """achieved GB/s as a fraction of the measured copy rate and of the nominal 8 TB/s (SURVEY 8(d) asks for both)"""
    return {"hbm_gbs": round(gbs, 1), "hbm_frac": round(gbs / peak, 4), "hbm_frac_nominal": round(gbs / NOMINAL_HBM_GBS, 4)}


def cpu_info():
    model = "unknown"
    try:
        for line in open("/proc/cpuinfo"):
            if line.startswith("model name"):
                model = line.split(":", 1)[1].strip()
                break
    except OSError:
        pass
    return {"nproc": os.cpu_count(), "affinity": len(os.sched_getaffinity(0)), "cpu_model": model,
            "oracle_flags": "gcc -O2 -ffp-contract=off -fopenmp"}


def ncu_traffic(kernel, workload):
    """DRAM bytes per launch of `kernel` on `workload` from the committed ncu capture (profiles/r2_ncu_kernels.csv:
    dram__bytes_read.sum + dram__bytes_write.sum of one --set full capture).  None when no capture of exactly this
    kernel instantiation and workload is on file: the number is evidence of a capture, never an estimate."""
    path = os.path.join(ROOT, "profiles", "r2_ncu_kernels.csv")
    try:
        import csv
        for row in csv.DictReader(open(path)):
            if row["kernel"] == kernel and row["workload"] == workload:
                return float(row["dram_read_bytes"]) + float(row["dram_write_bytes"]), "profiles/r2_ncu_kernels.csv: " + row["capture"]
    except (OSError, KeyError, ValueError):
        pass
    return None, None


class ClockSampler:
    """nvidia-smi clocks / throttle reasons sampled DURING the timed region."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
         "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, index):
        self.p = None
        try:
            self.p = subprocess.Popen(["nvidia-smi", "-i", str(index), f"--query-gpu={self.Q}", "--format=csv,noheader,nounits",
                                       "-lms", "20"], stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
        except Exception:
            pass

    def stop(self):
        if self.p is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        time.sleep(0.15)
        self.p.terminate()
        out = self.p.communicate()[0]
        sm, mx, reasons = [], [], set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for line in out.strip().splitlines():
            c = [v.strip() for v in line.split(",")]
            if len(c) < 7:
                continue
            try:
                sm.append(float(c[0])); mx.append(float(c[1]))
            except ValueError:
                continue
            for nme, v in zip(names, c[3:7]):
                if v.lower().startswith("active"):
                    reasons.add(nme)
        return {"sm_mhz": float(np.median(sm)) if sm else None, "sm_max_mhz": max(mx) if mx else None,
                "samples": len(sm), "reasons": sorted(reasons)}


# ----------------------------------------------------------------------------- workloads
def make_cfg4(small=False):
    import workloads as W
    if small:
        return W.cfg4_shear(seed=4, n=128, n_part=2500, R=4.0)
    return W.cfg4_shear()


def coupled_bytes_per_step(n_cells):
    """Algorithmic HBM bytes of the dominant (PSM stream-collide) kernel per launch, DESIGN.md section 7:
    19 populations read + 19 written (304 B) + the 8-byte solid slot read, per cell."""
    return 312.0 * n_cells


def dem_bytes(passes, n, ends):
    """Algorithmic HBM bytes per step of each DEM kernel group: per particle, plus per contact
    END in the contact group (every contact has two ends; `ends` = 2 x contacts + wall contacts)."""
    per_particle = {
        "dem_keys": 48 + 32 + 96 + 96 + 32 + 48 + 8,   # kick of the previous step + drift + keys in one pass: sums, (x,R), v w a
                                                       # alpha read; v w a alpha, (x,R), predictor, key + home index written
        "dem_sort": 4 + 16 * passes,                   # histogram read + (key, index) read and written per pass
        "dem_gather": 8 + 4 + 4 + 4 + 32 + 32 + 16 + 12,   # keys, indices, ids (ranges + rank); (x,R) read; (x,R), fp32 copy, id, index, counter written
        "dem_contact": 4 + 32 + 16 + 8 + 4 + 8}        # detect: key, own records; scan: two counters read, offset written; fill: row descriptor
    per_end = {"dem_contact": 4 + 4                    # detect: the entry written, fill: read
                              + 4 + 24                 # fill: partner's id + 6 words of end records written (owner, partner, home indices, previous end, id)
                              + 20 + 24 + 24           # force: end records read, previous delta_t read, new delta_t written
                              + (32 + 48) / 2.0}       # force: the owner's (x,R) + predictor once per particle ~ half an end's share; partners come from L2
    out = {k: v * n for k, v in per_particle.items()}
    out["dem_contact"] += per_end["dem_contact"] * ends + 48.0 * min(n, ends)   # + the sums of every particle in contact written
    return out, per_particle, per_end


def paper_bed_runs(args, timed, peak, warm, steps, precisions):
    import torch
    import paper_2512_04997_b200 as L
    from paper_2512_04997_b200 import Coupled, Dem, Lbm
    import workloads as W
    bed = {}
    for prec in precisions:
        bpc = 312.0 if prec == "f64" else 160.0
        for phi in (0.0, 0.15, 0.30, 0.45):
            lbb, cpb, pdb, xb, vb, wb, Rb = W.paper_bed(phi, contacts=True)
            glb = Lbm(lbb, precision=prec)
            gdb = Dem(pdb, xb, vb, wb, Rb)
            gb = Coupled(glb, gdb, cpb, 10.0)
            gb.step(warm); torch.cuda.synchronize()
            L.ledds_profile(True)
            msb = timed(gb.step, steps) / steps
            prb = {nm: round(L.ledds_profile_read(i)[0] / steps, 5) for i, nm in enumerate(L.KERNEL_GROUPS)}
            L.ledds_profile(False)
            q = torch.zeros(4, dtype=torch.int32, device="cuda")
            if len(Rb):
                L.ledds_dem_query(gdb.h, gdb.history, gdb.scratch, None, None, None, None, 0, q, None, None)
            ncb = int(np.prod(lbb["shape"]))
            bed["%s phi=%.2f" % (prec, phi)] = {
                "spheres": len(Rb), "solid_fraction": round(len(Rb) * 4.0 / 3.0 * np.pi * 1e3 / ncb, 4), "contacts": int(q[0].item()),
                "mlups": round(ncb / msb / 1e3, 1), "ms_per_step": round(msb, 4), "kernel_ms_per_step": prb,
                "step": fracs(bpc * ncb / msb / 1e6, peak), "lbm_kernel": fracs(bpc * ncb / prb["lbm"] / 1e6, peak),
                "status_word": int(gdb.status[0].item())}
            del gb, gdb, glb
            torch.cuda.empty_cache()
    bed["protocol"] = f"{warm} warm-up + {steps} timed LBM steps (the paper: 500 + 2500, PAPER.md:876)"
    bed["note"] = ("80 M cells (24.3 GB of fp64 populations), TRT, n_sub = 10; periodic x, y and walls in z instead of the paper's "
                   "inlet/outlet; columns of touching spheres; the paper reports this workload only as figures (A100-SXM4 80 GB)")
    return bed


def max_over_ranks(ms, world, device="cuda"):
    """Elapsed time of the slowest rank (replicas run independently; the job is as slow as the slowest)."""
    if world <= 1:
        return float(ms)
    import torch
    import torch.distributed as dist
    t = torch.tensor([ms], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def whole_job_mlups(n_cells, ms_step, world):
    """Cells updated per second by all replicas together, in 1e6."""
    return world * n_cells / ms_step / 1e3


def run_ours(args, rank, world):
    import torch
    import torch.distributed as dist
    import paper_2512_04997_b200 as L
    from paper_2512_04997_b200 import Coupled, Dem, Lbm
    import workloads as W

    local = int(os.environ.get("LOCAL_RANK", 0))
    torch.cuda.set_device(local)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))
    K, Wm = args.steps, args.warmup
    peak, peak_src = peaks()
    launches0 = L.ledds_launch_count()

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    def timed(fn, k):
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        barrier()
        e0.record(); fn(k); e1.record()
        barrier()
        return max_over_ranks(e0.elapsed_time(e1), world)

    out = {}
    # ------------------------------------------------------------------ main: coupled step, configs[3]
    small = args.workload == "small"
    lbm, cpl, pd, x, v, w, R, u = make_cfg4(small)
    n_cells = int(np.prod(lbm["shape"])); n_part = len(R)
    g_lbm = Lbm(lbm, None, u)
    g_dem = Dem(pd, x, v, w, R)
    g = Coupled(g_lbm, g_dem, cpl, float(R.max()))
    g.step(Wm)
    torch.cuda.synchronize()
    sampler = ClockSampler(local) if rank == 0 else None
    L.ledds_profile(True)
    l0 = L.ledds_launch_count()
    ms = timed(g.step, K)
    launches = L.ledds_launch_count() - l0
    prof = {name: L.ledds_profile_read(i) for i, name in enumerate(L.KERNEL_GROUPS)}
    L.ledds_profile(False)
    clocks = sampler.stop() if sampler else None
    status = int(g_dem.status[0].item())
    ms_step = ms / K
    mlups = whole_job_mlups(n_cells, ms_step, world)
    k_ms, k_n = prof["lbm"]
    k_ms_avg = k_ms / max(k_n, 1)
    bytes_launch = coupled_bytes_per_step(n_cells)
    achieved = bytes_launch / (k_ms_avg * 1e-3) / 1e9 if k_ms_avg > 0 else 0.0
    PSM_KERNEL = "lbm_psm_kernel<double, unsigned int, 128, false, false>"
    traffic, traffic_src = ncu_traffic(PSM_KERNEL, "configs[3]") if not small else (None, None)
    out.update({
        "metric": METRIC, "value": round(mlups, 1), "unit": "MLUPS", "n_gpus": world, "steps": K, "warmup": Wm,
        "ms_per_step": round(ms_step, 5), "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
        "dtype": "f64", "data": "synthetic",
        "config": {"workload": "configs[3] coupled shear: 256^3 D3Q19 BGK tau=0.6, periodic xy, walls z +-0.05, "
                               "20000 spheres R=4 (RSA seed 4), PSM coupling, n_sub=1" if not small else
                               "SMALL stand-in (128^3, 2500 spheres) -- not the headline configuration",
                   "lattice": list(lbm["shape"]), "particles": n_part, "l2": "inputs exceed L2 (5.1 GB of populations)",
                   "parallelism": "replicas only" if world > 1 else "1 GPU"},
        "coupled_steps_per_s": round(world * 1e3 / ms_step, 2),
        "particle_updates_per_s": round(world * n_part * cpl["n_sub"] * 1e3 / ms_step, 1),
        "gpu_launches": int(launches),
        "status_word": status,
        "kernel_ms_per_step": {k: round(vv[0] / K, 5) for k, vv in prof.items()},
        "kernel_ms_note": "dem_sort/gather/contact run on a side stream beside cpl_raster and lbm: their event spans overlap those",
        "roofline": {"bound": "hbm", "kernel": PSM_KERNEL, "achieved": round(achieved, 1), "peak": peak,
                     "peak_source": peak_src, "unit": "GB/s", "frac": round(achieved / peak, 4),
                     "frac_nominal": round(achieved / NOMINAL_HBM_GBS, 4), "peak_nominal": NOMINAL_HBM_GBS,
                     "bytes_per_launch": bytes_launch, "kernel_ms": round(k_ms_avg, 5),
                     "share_of_step": round(k_ms_avg / ms_step, 4), "traffic": traffic, "traffic_source": traffic_src},
        "clocks": clocks,
    })

    # ------------------------------------------------------------------ e2e through the public API with HOST buffers
    # per step: every input of ledds_coupled_step from pinned host memory (populations, particle state, last
    # hydrodynamic forces), the call, and every output back to the host (the UPDATED populations, particle state,
    # hydrodynamic force and torque)
    if rank == 0 or world > 1:
        e2e_steps = max(1, min(K, args.e2e_steps))
        f_host = torch.empty(19 * n_cells, dtype=torch.float64).pin_memory()
        f_out = torch.empty(19 * n_cells, dtype=torch.float64).pin_memory()
        f_dev_view = torch.empty(19 * n_cells, dtype=torch.float64, device="cuda")
        L.ledds_lbm_export(g_lbm.h, g_lbm.f, f_dev_view, None, None)
        f_host.copy_(f_dev_view); torch.cuda.synchronize()
        hp = {k: getattr(g_dem, k).cpu().pin_memory() for k in ("x", "v", "w", "a", "alpha", "radius")}
        hp["f_hyd"] = g.f_hyd.cpu().pin_memory(); hp["m_hyd"] = g.m_hyd.cpu().pin_memory()
        res = {k: torch.empty_like(hp[k]).pin_memory() for k in ("x", "v", "w", "a", "alpha", "f_hyd", "m_hyd")}
        h2d = f_host.numel() * 8 + sum(t.numel() * 8 for t in hp.values())
        d2h = f_out.numel() * 8 + sum(t.numel() * 8 for t in res.values())

        def e2e(k):
            for _ in range(k):
                f_dev_view.copy_(f_host, non_blocking=True)
                L.ledds_lbm_import(g_lbm.h, g_lbm.f, f_dev_view)
                for kk in ("x", "v", "w", "a", "alpha", "radius"):
                    getattr(g_dem, kk).copy_(hp[kk], non_blocking=True)
                g.f_hyd.copy_(hp["f_hyd"], non_blocking=True); g.m_hyd.copy_(hp["m_hyd"], non_blocking=True)
                g.step(1)
                L.ledds_lbm_export(g_lbm.h, g_lbm.f, f_dev_view, None, None)
                f_out.copy_(f_dev_view, non_blocking=True)
                for kk in ("x", "v", "w", "a", "alpha"):
                    res[kk].copy_(getattr(g_dem, kk), non_blocking=True)
                res["f_hyd"].copy_(g.f_hyd, non_blocking=True); res["m_hyd"].copy_(g.m_hyd, non_blocking=True)
                torch.cuda.current_stream().synchronize()
        e2e(1)
        ms_e = timed(e2e, e2e_steps) / e2e_steps
        out["e2e"] = {"value": round(world * n_cells / ms_e / 1e3, 1), "unit": "MLUPS", "ms_per_step": round(ms_e, 4),
                      "steps": e2e_steps, "h2d_bytes_per_step": int(h2d), "d2h_bytes_per_step": int(d2h),
                      "what": "per step: populations + particle state + last F_sf, M_sf from pinned host -> ledds_coupled_step -> "
                              "updated populations + particle state + F_sf, M_sf back to pinned host (PCIe-bound by construction)"}
        del f_host, f_out, f_dev_view
    del g, g_lbm, g_dem
    torch.cuda.empty_cache()

    # ------------------------------------------------------------------ sub-benchmarks (rank 0 of a 1-GPU run only)
    sub = {}
    if world == 1 and not args.no_sub:
        # configs[1]: LBM-only 128^3 TGV
        lb, rho, uu = W.cfg2_tgv(128 if not small else 64)
        gl = Lbm(lb, rho, uu)
        gl.step(20); torch.cuda.synchronize()
        ks = 1000 if not small else 100
        ms2 = timed(gl.step, ks) / ks
        nc2 = int(np.prod(lb["shape"]))
        _, r2, u2 = gl.export(want_moments=True)
        sub["cfg2_lbm_tgv128"] = {"mlups": round(nc2 / ms2 / 1e3, 1), "ms_per_step": round(ms2, 5), "steps": ks,
                                   **fracs(304.0 * nc2 / ms2 / 1e6, peak),
                                   "note": "638 MB of populations (> 126 MB L2); 304 B/cell"}
        del gl
        # the same with the TRT collision (Eq. 29-31), the model of the paper's own results
        gt = Lbm(dict(lb, collision=1), rho, uu)
        gt.step(20); torch.cuda.synchronize()
        ms2t = timed(gt.step, ks) / ks
        sub["cfg2_lbm_tgv128_trt"] = {"mlups": round(nc2 / ms2t / 1e3, 1), "ms_per_step": round(ms2t, 5), "steps": ks,
                                       **fracs(304.0 * nc2 / ms2t / 1e6, peak)}
        del gt
        # fp32 variant of the plain LBM path (152 B/cell), at 128^3 and at the headline lattice size
        if not args.sub_large_only:
            for nn in ((128, 256) if not small else (64,)):
                lbf, rhof, uuf = W.cfg2_tgv(nn)
                ncf = int(np.prod(lbf["shape"]))
                for prec, bpc in (("f32", 152.0), ("f64", 304.0)):
                    if prec == "f64" and nn == 128:
                        continue                                         # that is cfg2_lbm_tgv128 above
                    gf = Lbm(lbf, rhof, uuf, precision=prec)
                    gf.step(20); torch.cuda.synchronize()
                    kf = 400 if not small else 100
                    msf = timed(gf.step, kf) / kf
                    sub[f"lbm_tgv{nn}_{prec}"] = {"mlups": round(ncf / msf / 1e3, 1), "ms_per_step": round(msf, 5), "steps": kf,
                                                  **fracs(bpc * ncf / msf / 1e6, peak), "dtype": prec}
                    del gf
        # the paper's own validation combination on the headline workload: TRT collision (Eq. 29-31) + subdivision
        # solid fraction (Eq. 38, 10^3 points per cell)
        if not args.sub_large_only:
            lbv, cpv, pdv, xv, vv, wv, Rv, uv = make_cfg4(small)
            glv = Lbm(dict(lbv, collision=1), None, uv); gdv = Dem(pdv, xv, vv, wv, Rv)
            gv = Coupled(glv, gdv, dict(cpv, solid_fraction=1), float(Rv.max()))
            gv.step(3); torch.cuda.synchronize()
            L.ledds_profile(True)
            msv = timed(gv.step, 10) / 10
            prv = {nm: round(L.ledds_profile_read(i)[0] / 10, 5) for i, nm in enumerate(L.KERNEL_GROUPS) if nm in ("lbm", "cpl_raster", "cpl_reduce")}
            L.ledds_profile(False)
            ncv = int(np.prod(lbv["shape"]))
            sub["cfg4_trt_subdivision"] = {"mlups": round(ncv / msv / 1e3, 1), "ms_per_step": round(msv, 5), "steps": 10,
                                           "kernel_ms_per_step": prv, "status_word": int(gdv.status[0].item()),
                                           "note": "TRT + Eq. 38 with 1000 points per cell: the raster counts points for every boundary cell"}
            del gv, glv, gdv
            torch.cuda.empty_cache()
            # the headline workload on an fp32 lattice (ledds_coupled_step_f32): 160 B per cell
            glf = Lbm(lbv, None, uv.astype(np.float32), precision="f32"); gdf = Dem(pdv, xv, vv, wv, Rv)
            gf4 = Coupled(glf, gdf, cpv, float(Rv.max()))
            gf4.step(3); torch.cuda.synchronize()
            L.ledds_profile(True)
            msf4 = timed(gf4.step, 20) / 20
            prf = {nm: round(L.ledds_profile_read(i)[0] / 20, 5) for i, nm in enumerate(L.KERNEL_GROUPS) if nm in ("lbm", "cpl_raster", "cpl_reduce")}
            L.ledds_profile(False)
            sub["cfg4_f32_lattice"] = {"mlups": round(ncv / msf4 / 1e3, 1), "ms_per_step": round(msf4, 5), "steps": 20, "dtype": "f32 lattice, f64 solids and DEM",
                                       "kernel_ms_per_step": prf, **fracs(160.0 * ncv / prf["lbm"] / 1e6, peak),
                                       "status_word": int(gdf.status[0].item())}
            del gf4, glf, gdf
            torch.cuda.empty_cache()
        # the paper's own performance workload: 500 x 200 x 800 cells, spheres of
        # 20 cells diameter at solid fraction 0 ... 0.45, 10 DEM sub-steps per LBM step, TRT, distance-based fraction.  The
        # bed is packed so that the spheres touch (contacts = True): the DEM contact path is loaded.  Default: 5 warm-up +
        # 20 timed steps (a deviation from the paper's protocol, stated in the output); --paper-protocol runs the paper's
        # 500 + 2500 iterations on the fp64 and on the fp32 lattice.
        if not args.sub_large_only and not small:
            sub["paper_bed_500x200x800"] = paper_bed_runs(args, timed, peak, 5, 20, ("f64",))
            if args.paper_protocol:
                sub["paper_bed_500x200x800_paper_protocol"] = paper_bed_runs(args, timed, peak, 500, 2500, ("f64", "f32"))
        # configs[0] and configs[2]: small, launch-latency-bound workloads, timed plainly and replayed from a CUDA
        # graph (the library only enqueues on the caller's stream, so its calls can be captured)
        small_cfgs = not args.sub_large_only
        def graph_time(step_fn, per_graph, replays):
            side = torch.cuda.Stream()
            side.wait_stream(torch.cuda.current_stream())
            with torch.cuda.stream(side):
                step_fn(per_graph)                                  # warm-up on the capture stream
            torch.cuda.current_stream().wait_stream(side)
            torch.cuda.synchronize()
            gr = torch.cuda.CUDAGraph()
            with torch.cuda.graph(gr):
                step_fn(per_graph)
            gr.replay(); torch.cuda.synchronize()
            return timed(lambda k: [gr.replay() for _ in range(k)], replays) / (replays * per_graph)
        if small_cfgs:
            pd1, x1, v1, w1, R1 = W.cfg1_gas()
            g1 = Dem(pd1, x1, v1, w1, R1)
            g1.step(50); torch.cuda.synchronize()
            ms1 = timed(g1.step, 1000) / 1000
            try:
                ms1g = graph_time(g1.step, 20, 50)
            except Exception:                                           # a capture failure must not take the line down
                ms1g = float("nan")
            sub["cfg1_dem_gas_2048"] = {"steps_per_s": round(1e3 / ms1, 1), "particle_updates_per_s": round(len(R1) * 1e3 / ms1, 1),
                                         "cuda_graph_steps_per_s": round(1e3 / ms1g, 1),
                                         "cuda_graph_particle_updates_per_s": round(len(R1) * 1e3 / ms1g, 1),
                                         "status_word": int(g1.status[0].item()),
                                         "note": "one launch per step: a cluster of 8 blocks does the whole step (n <= 4096)"}
            del g1
            g1c = Dem(dict(pd1, no_single_block=1), x1, v1, w1, R1)     # the chain of kernels larger systems take, for comparison
            g1c.step(50); torch.cuda.synchronize()
            ms1c = timed(g1c.step, 1000) / 1000
            sub["cfg1_dem_gas_2048"]["kernel_chain_steps_per_s"] = round(1e3 / ms1c, 1)
            del g1c
            lb3, cp3, pd3, x3, v3, w3, R3 = W.cfg3_settling()
            gl3 = Lbm(lb3); gd3 = Dem(pd3, x3, v3, w3, R3); g3 = Coupled(gl3, gd3, cp3, float(R3.max()))
            g3.step(20); torch.cuda.synchronize()
            ms3 = timed(g3.step, 500) / 500
            try:
                ms3g = graph_time(g3.step, 20, 25)                      # an even number of steps per graph keeps the lattice parity
            except Exception:
                ms3g = float("nan")
            nc3 = int(np.prod(lb3["shape"]))
            sub["cfg3_settling_64x64x256"] = {"coupled_steps_per_s": round(1e3 / ms3, 1), "mlups": round(nc3 / ms3 / 1e3, 1),
                                               "cuda_graph_coupled_steps_per_s": round(1e3 / ms3g, 1),
                                               "cuda_graph_mlups": round(nc3 / ms3g / 1e3, 1), "status_word": int(gd3.status[0].item()),
                                               "note": "159 MB per lattice: close to L2 size, so MLUPS may exceed the HBM bound"}
            del g3, gl3, gd3
        # configs[4]: DEM-only, 4 M polydisperse spheres (jittered-lattice placement), + supplementary dense state
        for name, dense, prec in (("cfg5_dem_pour_4M", False, "f64"), ("cfg5_dense_supplement_4M", True, "f64"),
                                  ("cfg5_dem_pour_4M_f32", False, "f32"), ("cfg5_dense_supplement_4M_f32", True, "f32")):
            pd5, x5, v5, w5, R5 = W.cfg5_pour(n_side=160 if not small else 40, n_part=4_000_000 if not small else 64000, dense=dense)
            gd = Dem(pd5, x5, v5, w5, R5, precision=prec)
            gd.step(5); torch.cuda.synchronize()
            L.ledds_profile(True)
            kd = 50
            ms5 = timed(gd.step, kd) / kd
            pr = {nm: round(L.ledds_profile_read(i)[0] / kd, 5) for i, nm in enumerate(L.KERNEL_GROUPS) if nm.startswith("dem")}
            L.ledds_profile(False)
            q = torch.zeros(4, dtype=torch.int32, device="cuda")
            (L.ledds_dem_query_f32 if prec == "f32" else L.ledds_dem_query)(gd.h, gd.history, gd.scratch, None, None, None, None, 0, q, None, None)
            contacts = int(q[0].item())
            ncell = 1
            for a in range(3):
                ncell *= max(1, int((pd5["hi"][a] - pd5["lo"][a]) / pd5["cell"]))
            ends = 2 * contacts                                          # wall contacts (one end each) are counted as two: < 1 % here
            bytes_k, bpp, bpe = dem_bytes((max(1, int(np.ceil(np.log2(ncell)))) + 7) // 8, len(R5), ends)
            gbs = {nm: fracs(bytes_k[nm] / (pr[nm] * 1e-3) / 1e9, peak) for nm in bytes_k if pr.get(nm, 0) > 0}
            total_bytes = sum(bytes_k.values())
            if prec == "f32":                                            # the fp64 byte model does not apply: times only
                sub[name] = {"particle_updates_per_s": round(len(R5) * 1e3 / ms5, 1), "ms_per_step": round(ms5, 5), "steps": kd,
                             "particles": len(R5), "contacts": contacts, "kernel_ms_per_step": pr, "dtype": "f32",
                             "status_word": int(gd.status[0].item())}
                del gd
                torch.cuda.empty_cache()
                continue
            sub[name] = {"particle_updates_per_s": round(len(R5) * 1e3 / ms5, 1), "ms_per_step": round(ms5, 5), "steps": kd,
                         "particles": len(R5), "contacts": contacts, "kernel_ms_per_step": pr,
                         "algorithmic_bytes_per_particle": bpp, "algorithmic_bytes_per_contact_end": bpe, "kernel_hbm": gbs,
                         "pipeline": fracs(total_bytes / (ms5 * 1e-3) / 1e9, peak),
                         "note": "one call of 50 steps: import (caller order -> home order) and export are inside the timed call, "
                                 "their kernels are not in any group of kernel_ms_per_step",
                         "status_word": int(gd.status[0].item())}
            del gd
            torch.cuda.empty_cache()
        out["sub"] = sub
    out["gpu_launches_total"] = int(L.ledds_launch_count() - launches0)
    if world > 1:
        dist.destroy_process_group()
    return out


# ----------------------------------------------------------------------------- oracle legs
# The CPU baseline of SURVEY 8(d) / BASELINE.md section 3: the oracle as it stands, timed on the host cores of the GPU
# box on a bounded sample of each config, once with all cores (OpenMP) and once with OMP_NUM_THREADS=1.  Every leg runs
# in a process of its own (the thread count is fixed when liboracle.so loads); that process imports oracle/ and
# workloads/ only, never the CUDA library.
ORACLE_LEGS = {
    # name: (steps with all cores, steps single-threaded)
    "cfg1": (10, 10), "cfg2": (20, 5), "cfg3": (5, 2), "cfg4": (2, 1), "cfg5": (2, 2),
}


def oracle_leg(name, steps, small=False):
    """Runs one leg in THIS process; returns its record."""
    import oracle
    import workloads as W
    threads = int(os.environ.get("OMP_NUM_THREADS", "0")) or len(os.sched_getaffinity(0))
    rec = {"leg": name, "steps": steps, "kind": "oracle"}
    if name == "cfg1":
        pd, x, v, w, R = W.cfg1_gas()
        d = oracle.Dem(pd, x, v, w, R)
        d.step(1)
        t0 = time.perf_counter(); d.step(steps); dt = time.perf_counter() - t0
        rec.update(value=round(len(R) * steps / dt, 1), unit="particle-updates/s", steps_per_s=round(steps / dt, 2), cores=1,
                   sample=f"{steps} oracle DEM steps of configs[0] (2048 spheres) after one untimed step; the DEM oracle is single-threaded")
    elif name == "cfg2":
        lb, rho, u = W.cfg2_tgv(128 if not small else 48)
        f = oracle.lbm_equilibrium(lb["shape"], rho, u)
        f = oracle.lbm_run(lb["shape"], f, lb["tau"], 1)
        t0 = time.perf_counter(); oracle.lbm_run(lb["shape"], f, lb["tau"], steps); dt = time.perf_counter() - t0
        n = int(np.prod(lb["shape"]))
        rec.update(value=round(n * steps / dt / 1e6, 3), unit="MLUPS", cores=threads,
                   sample=f"{steps} oracle LBM steps of configs[1] ({lb['shape'][0]}^3 Taylor-Green) after one untimed step")
    elif name in ("cfg3", "cfg4"):
        if name == "cfg3":
            lbm, cpl, pd, x, v, w, R = W.cfg3_settling() if not small else W.cfg3_settling(shape=(32, 32, 64), R=5.0, z0=40.0)
            u = None
        else:
            lbm, cpl, pd, x, v, w, R, u = make_cfg4(small)
        oc = oracle.Coupled(lbm, cpl, oracle.Dem(pd, x, v, w, R), oracle.lbm_equilibrium(lbm["shape"], None, u))
        oc.step(1)
        t0 = time.perf_counter(); oc.step(steps); dt = time.perf_counter() - t0
        n = int(np.prod(lbm["shape"]))
        rec.update(value=round(n * steps / dt / 1e6, 3), unit="MLUPS", coupled_steps_per_s=round(steps / dt, 4), cores=threads,
                   sample=f"{steps} coupled oracle steps of {'configs[2]' if name == 'cfg3' else 'configs[3]'} "
                          f"({n} cells, {len(R)} spheres) after one untimed step")
    elif name == "cfg5":
        n_side, n_part = (100, 1_000_000) if not small else (30, 27000)
        pd, x, v, w, R = W.cfg5_pour(n_side=n_side, n_part=n_part)
        d = oracle.Dem(pd, x, v, w, R)
        t0 = time.perf_counter(); d.step(steps); dt = time.perf_counter() - t0
        rec.update(value=round(len(R) * steps / dt, 1), unit="particle-updates/s", cores=1,
                   sample=f"{steps} oracle DEM steps of a quarter-size configs[4] state ({n_part} spheres, same density and parameters; the "
                          "rate per particle does not depend on the size); the DEM oracle is single-threaded")
    else:
        raise ValueError(name)
    return rec


def oracle_leg_subprocess(name, threads, small):
    """-> record of one leg run in a child process with the given OpenMP thread count (None = all cores)"""
    env = dict(os.environ)
    if threads:
        env["OMP_NUM_THREADS"] = str(threads)
    else:
        env.pop("OMP_NUM_THREADS", None)
    cmd = [sys.executable, os.path.abspath(__file__), "--oracle-leg", name, "--oracle-leg-threads", str(threads or 0)]
    if small:
        cmd += ["--workload", "small"]
    try:
        r = subprocess.run(cmd, env=env, capture_output=True, text=True, timeout=600)
        for line in reversed(r.stdout.strip().splitlines()):
            if line.startswith("{"):
                return json.loads(line)
        return {"leg": name, "error": (r.stderr or r.stdout)[-300:]}
    except Exception as e:                                      # a baseline leg must never take the bench line down
        return {"leg": name, "error": repr(e)}


def cpu_baselines(small):
    """all legs, all cores and one thread; the main entry (configs[3], all cores) is the line's cpu_baseline"""
    legs = {}
    for name in ORACLE_LEGS:
        legs[name] = {"all_cores": oracle_leg_subprocess(name, None, small)}
        if name in ("cfg2", "cfg3", "cfg4"):                     # the DEM oracle has no OpenMP loop: one run says it all
            legs[name]["one_thread"] = oracle_leg_subprocess(name, 1, small)
    return legs


def build_oracle_only():
    import importlib.util
    spec = importlib.util.spec_from_file_location("_oracle_build", os.path.join(ROOT, "oracle", "build.py"))
    m = importlib.util.module_from_spec(spec)
    spec.loader.exec_module(m)
    m.build()


def run_reference(args, rank, world):
    """The reference arm of this tier: the oracle alone on the host cores.  Imports oracle/ and workloads/ only."""
    if rank != 0:
        return None
    K, Wm = args.steps, args.warmup
    # one coupled oracle step of the full configs[3] state takes ~1 s on 16 cores: the full state whenever the run fits
    # ~3 minutes, else a 1/8-volume stand-in of the same solid fraction and parameters (and the line says so)
    small = (K + Wm) > 150 or args.workload == "small"
    import oracle
    lbm, cpl, pd, x, v, w, R, u = make_cfg4(small)
    n_cells = int(np.prod(lbm["shape"]))
    f0 = oracle.lbm_equilibrium(lbm["shape"], None, u)
    oc = oracle.Coupled(lbm, cpl, oracle.Dem(pd, x, v, w, R), f0)
    oc.step(Wm)
    t0 = time.perf_counter()
    oc.step(K)
    ms_step = (time.perf_counter() - t0) * 1e3 / K
    cores = len(os.sched_getaffinity(0))
    mlups = n_cells / ms_step / 1e3
    sample = ("each step = one coupled oracle step of the full configs[3] state" if not small else
              "each step = one coupled oracle step of a 1/8-volume stand-in (128^3, 2500 spheres, same solid fraction "
              "and parameters); MLUPS is size-independent, steps/s is scaled by 1/8")
    return {"impl": "reference", "metric": METRIC, "value": round(mlups, 3), "unit": "MLUPS", "n_gpus": world, "steps": K,
            "warmup": Wm, "ms_per_step": round(ms_step, 3), "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
            "dtype": "f64", "data": "synthetic", "same_config": not small,
            "config": {"workload": "configs[3] coupled shear (CPU oracle, oracle/*.c, gcc -O2 -ffp-contract=off -fopenmp)"
                                   if not small else "SMALL stand-in of configs[3] (128^3, 2500 spheres) -- not the headline configuration",
                       "lattice": list(lbm["shape"]), "particles": len(R)},
            "cpu_baseline": {"value": round(mlups, 3), "unit": "MLUPS", "cores": cores, "kind": "oracle", "sample": sample, **cpu_info()},
            "e2e": {"value": round(mlups, 3), "unit": "MLUPS", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0}}


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=50)
    ap.add_argument("--warmup", type=int, default=5)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--workload", default="cfg4", choices=["cfg4", "small"])
    ap.add_argument("--e2e-steps", type=int, default=5)
    ap.add_argument("--no-sub", action="store_true")
    ap.add_argument("--sub-large-only", action="store_true", help="skip the latency-bound small configs (profiling of the 4 M DEM kernels)")
    ap.add_argument("--no-cpu", action="store_true")
    ap.add_argument("--paper-protocol", action="store_true", help="also run the paper's bed with its 500 + 2500 iterations, fp64 and fp32")
    ap.add_argument("--oracle-leg", default=None, help="internal: time one oracle leg in this process and print its JSON")
    ap.add_argument("--oracle-leg-threads", type=int, default=0)
    args = ap.parse_args()
    rank = int(os.environ.get("RANK", 0)); world = int(os.environ.get("WORLD_SIZE", 1))
    if args.oracle_leg:                                           # child process of cpu_baselines(): oracle/ only
        build_oracle_only()
        steps = ORACLE_LEGS[args.oracle_leg][1 if args.oracle_leg_threads == 1 else 0]
        print(json.dumps(oracle_leg(args.oracle_leg, steps, args.workload == "small")), flush=True)
        return
    if args.impl == "reference":                                  # the oracle alone: the CUDA library is neither built nor loaded
        if rank == 0:
            build_oracle_only()
            print(json.dumps(run_reference(args, rank, world)), flush=True)
        return
    args.warmup = max(args.warmup, 3)
    import fcntl
    import __graft_entry__ as ge
    with open(os.path.join(ROOT, ".build.lock"), "w") as lock:    # one rank builds, the others find the libraries up to date
        fcntl.flock(lock, fcntl.LOCK_EX)
        ge.build()
        fcntl.flock(lock, fcntl.LOCK_UN)
    out = run_ours(args, rank, world)
    if rank == 0:
        if world == 1 and not args.no_cpu:
            legs = cpu_baselines(args.workload == "small")
            main_leg = legs.get("cfg4", {}).get("all_cores", {})
            out["cpu_baseline"] = {"value": main_leg.get("value"), "unit": "MLUPS", "cores": main_leg.get("cores"), "kind": "oracle",
                                   "sample": main_leg.get("sample", main_leg.get("error")), **cpu_info(), "legs": legs}
        print(json.dumps(out), flush=True)


if __name__ == "__main__":
    main()
