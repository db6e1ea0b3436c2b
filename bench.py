#!/usr/bin/env python
"""bench.py -- one SCF step of the hot path (nao_geneig + nao_fermi_mu + nao_density_matrix) on synthetic NAO-shaped
matrices (BASELINE.json configs), timed on the device with CUDA events.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--workload c2|c3|c1|c0|c4] [--impl ours|reference]

A "step" is one pass of the whole path over one batch: factor S, reduce, tridiagonalise, divide-and-conquer,
back-transform, C = L^{-H} Z, Fermi level, density matrices.  Multi-GPU: the path does not shard (one matrix per
GPU, no collective) -- N ranks run N independent replicas ("replicas only"); time = max over ranks.
Prints ONE JSON line on rank 0.
"""
import argparse
import ctypes
import json
import os
import subprocess
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

WORKLOADS = {
    "c0": dict(idx=0, desc="config 0: 8-atom cluster, n=104 real, 1 item"),
    "c1": dict(idx=1, desc="config 1: 64-atom cell, n=832 complex, 8 k x 2 spins = 16 items"),
    "c2": dict(idx=2, desc="config 2: 512-atom collinear cell, n=6656 real, 2 spin channels"),
    "c3": dict(idx=3, desc="config 3: 384-atom noncollinear cell, 2N=9984 complex, S real 4992"),
    "c4": dict(idx=4, desc="config 4: 1024-atom noncollinear cell, 2N=26624 complex, S real 13312"),
}
FP64_DMMA_PEAK_TFLOPS = 148 * 128 * 1.965e9 / 1e12      # 148 SMs x 128 flop/clk/SM x 1.965 GHz = 37.2


def useful_flops(prob):
    """One-stage-equivalent real flop count of one step: potrf n^3/3, reduce n^3, tridiagonalise
    4n^3/3, D&C 4n^3/3 (real), back-transform 2n^3, L^{-H}Z n^3, DM n^3; complex flops count 4x (beta)."""
    n, beta = prob.n, (4.0 if prob.is_complex else 1.0)
    nS = prob.S.shape[-1]
    potrf = (1.0 if prob.nc_block_s else beta) * nS ** 3 / 3.0
    per_item = beta * n ** 3 * (1.0 + 4.0 / 3.0 + 2.0 + 1.0 + 1.0) + 4.0 / 3.0 * n ** 3
    return prob.batch * per_item + (1 if prob.nc_block_s else prob.batch) * potrf


class ClockSampler:
    """nvidia-smi clocks / throttle reasons sampled every 200 ms while the timed region runs."""

    def __init__(self, gpu_index):
        self.rows, self.proc, self.gpu = [], None, gpu_index

    def start(self):
        q = "clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown," \
            "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap"
        try:
            self.proc = subprocess.Popen(["nvidia-smi", "-i", str(self.gpu), "--query-gpu=" + q, "--format=csv,noheader,nounits",
                                          "-lms", "200"], stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.thread = threading.Thread(target=self._read, daemon=True)
            self.thread.start()
        except Exception:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.rows.append([x.strip() for x in line.split(",")])

    def stop(self):
        if self.proc is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        time.sleep(0.25)
        self.proc.terminate()
        try:
            self.proc.wait(timeout=2)
        except Exception:
            self.proc.kill()
        sm = sorted(float(r[0]) for r in self.rows if r and r[0].replace(".", "").isdigit())
        mx = [float(r[1]) for r in self.rows if len(r) > 1 and r[1].replace(".", "").isdigit()]
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        reasons = [nm for k, nm in enumerate(names) if any(len(r) > 3 + k and r[3 + k].lower().startswith("active") for r in self.rows)]
        return {"sm_mhz": sm[len(sm) // 2] if sm else None, "sm_max_mhz": max(mx) if mx else None, "reasons": reasons,
                "samples": len(sm)}


def oracle_sample(workload, budget_atoms=None):
    """The oracle, as it stands, on a bounded sample of the workload: the same recipe at a reduced atom count that
    the Jacobi oracle finishes in ~10-30 s; extrapolated to the full size by the N^3 law of Jacobi sweeps."""
    import oracle
    from paper_2606_09058_b200.synth import make_config, CONFIGS
    idx = WORKLOADS[workload]["idx"]
    full_nat = CONFIGS[idx]["nat"]
    nat = budget_atoms or {0: 8, 1: 16, 2: 64, 3: 32, 4: 32}[idx]
    prob = make_config(idx, nat=nat)
    t0 = time.time()
    oracle.solve_problem(prob)
    dt = time.time() - t0
    scale = (full_nat / float(nat)) ** 3
    cores = int(os.environ.get("OMP_NUM_THREADS", os.cpu_count() or 1))
    full_run = None
    if idx == 2:       # wall time of the one full run of this oracle at config 2, as recorded by the script that wrote the digest
        try:
            with open(os.path.join(ROOT, "tests", "golden", "c2_oracle_run.json")) as fh:
                full_run = json.load(fh)
        except Exception:
            full_run = None
    return dict(value=dt * scale, unit="s", cores=cores, kind="oracle", extrapolated=scale != 1.0, measured_s=dt, full_run=full_run,
                sample="%s recipe at %d atoms (n=%d, batch %d): %.2f s measured, x%.0f by the N^3 law to %d atoms"
                       % (workload, nat, prob.n, prob.batch, dt, scale, full_nat))


def oracle_in_run():
    """SURVEY.md 8d protocol: the Jacobi oracle timed in THIS run where it ends in seconds -- config 0 whole (geneig + Fermi +
    D), config 1 on two of its 16 items (eigensolve + D each; x8 for the batch, flagged as extrapolated)."""
    import numpy as np
    import oracle
    from paper_2606_09058_b200.synth import make_config
    cores = int(os.environ.get("OMP_NUM_THREADS", os.cpu_count() or 1))
    out = {}
    prob = make_config(0)
    t0 = time.time(); oracle.solve_problem(prob); dt = time.time() - t0
    out["c0"] = dict(value=dt, unit="s", cores=cores, kind="oracle", extrapolated=False,
                     sample="config 0 whole (n=%d, batch %d)" % (prob.n, prob.batch))
    prob = make_config(1)
    t0 = time.time()
    for b in (0, 9):
        e, C, _ = oracle.geneig(prob.H_full(b), prob.S_full(b))
        oracle.density(C, (e < np.median(e)).astype(np.float64))
    dt = time.time() - t0
    out["c1"] = dict(value=dt * prob.batch / 2.0, unit="s", cores=cores, kind="oracle", extrapolated=True, measured_s=dt,
                     sample="items 0 and 9 of %d measured (n=%d complex, eigensolve + density matrix): %.2f s, x%d"
                            % (prob.batch, prob.n, dt, prob.batch // 2))
    return out


def cpu_certificate_time(prob, E, C, ncols=512):
    """wall time of the CPU-side a-posteriori certificate (residual H C - S C diag(e) and C^H S C - I, numpy /
    host BLAS) for the eigenpairs the GPU returned, on a bounded sample of `ncols` evenly spaced eigenvectors; the products
    are linear in the number of columns, so the full-matrix time is the measured one x n / ncols (flagged)."""
    import numpy as np
    n = prob.n
    cols = np.linspace(0, n - 1, min(ncols, n)).astype(np.int64)
    Cs = np.ascontiguousarray(C[0][cols].cpu().numpy().T)            # stored row k = eigenvector k
    e = E[0].cpu().numpy()[cols]
    Hm, Sm = prob.H_full(0), prob.S_full(0)
    t0 = time.time()
    SC = Sm @ Cs
    R = Hm @ Cs - SC * e[None, :]
    G = Cs.conj().T @ SC
    G[np.diag_indices(len(cols))] -= 1.0
    resid, orth = float(np.abs(R).max()), float(np.abs(G).max())
    dt = time.time() - t0
    return dict(value=dt * n / len(cols), unit="s", cores=os.cpu_count(), kind="numpy certificate (residual + S-orthonormality)",
                extrapolated=True, measured_s=dt, max_residual=resid, max_orthonormality_defect=orth,
                sample="%d of %d eigenvectors measured: %.2f s, x%.1f" % (len(cols), n, dt, n / len(cols)))


def cpu_library_time(workload):
    """scipy.linalg.eigh(H, S) (LAPACK dsygvd/zhegvd on all host cores) on the FIRST item of the workload: a practical CPU
    time beside the (deliberately plain) Jacobi oracle (SURVEY.md 8d item ii).  An independent library, not the oracle and
    not the product path; only timed where it ends within about a minute (configs 0-2)."""
    import scipy.linalg as sl
    from paper_2606_09058_b200.synth import make_config
    idx = WORKLOADS[workload]["idx"]
    if idx > 2:
        return None
    prob = make_config(idx)
    t0 = time.time()
    sl.eigh(prob.H_full(0), prob.S_full(0), driver="gvd")
    dt = time.time() - t0
    return dict(value=dt * prob.batch, unit="s", cores=os.cpu_count(), kind="scipy.linalg.eigh (LAPACK gvd), eigenpairs only",
                sample="item 0 of %d measured: %.2f s; value = x%d items (no Fermi level, no density matrix)" % (prob.batch, dt, prob.batch))


def read_traffic(kernel, workload):
    """DRAM bytes per launch of `kernel` from the committed ncu captures (profiles/r03_traffic.csv, else r02_traffic.csv: one row per
    kernel and workload, written from `ncu --metrics dram__bytes_read.sum,dram__bytes_write.sum` over one whole step)."""
    import csv
    for name in ("r03_traffic.csv", "r02_traffic.csv"):      # the newest capture that has the row (the kernels did not change)
        try:
            with open(os.path.join(ROOT, "profiles", name)) as fh:
                for r in csv.DictReader(fh):
                    if r["kernel"] == kernel and r["workload"] == workload:
                        return float(r["dram_bytes_total"]) / max(1, int(r["launches"])), r["source"]
        except Exception:
            pass
    return None, None


def side_record(nao, torch, workload, dev, hbm_peak, dmma_meas, steps=3, warmup=2, groups=True, cpu_certificate=False,
                other_reduction=False):
    """A second workload timed in the same run (device-resident inputs, CUDA events, `warmup` + `steps` full steps, then one
    step with the library's event timers): ms per step, phases, and the rooflines of hetrd_panel_kernel / gemm_kernel."""
    from paper_2606_09058_b200.synth import make_config
    prob = make_config(WORKLOADS[workload]["idx"])
    flags = nao.NAO_NC_BLOCK_S if prob.nc_block_s else 0
    dt = nao.NAO_COMPLEX if prob.is_complex else nao.NAO_REAL
    H = torch.from_numpy(prob.H).to(dev); S0 = torch.from_numpy(prob.S).to(dev); S = torch.empty_like(S0)
    work = torch.empty(nao.geneig_workspace(prob.n, prob.batch, dt, flags) + 256, dtype=torch.uint8, device=dev)
    Dbuf = torch.empty_like(H)
    weights = [float(x) for x in prob.weights]
    in_bytes = H.numel() * H.element_size() + S0.numel() * S0.element_size()
    flush = None if in_bytes > (256 << 20) else torch.empty(256 << 20, dtype=torch.uint8, device=dev)

    last = {}

    def step():
        S.copy_(S0)
        E, C, info = nao.geneig(H, S, flags=flags, work=work)
        mu, F = nao.fermi_mu(E, weights, prob.n_electrons, prob.kT)
        nao.density_matrix(C, F, out=Dbuf)
        last["E"], last["C"] = E, C
        return info, mu
    for _ in range(warmup):
        info, mu = step()
    torch.cuda.synchronize()
    assert int(info.abs().max()) == 0
    ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    l0 = nao.launch_count()
    tot = 0.0
    for _ in range(steps):
        if flush is not None:
            flush.zero_()
        ev0.record(); step(); ev1.record(); torch.cuda.synchronize()
        tot += ev0.elapsed_time(ev1)
    ms = tot / steps
    launches = (nao.launch_count() - l0) // steps
    nao.profile_enable(True); step(); torch.cuda.synchronize()
    phases = nao.profile_read(); kp = nao.profile_kernel(0); kg = nao.profile_kernel(1)
    nao.profile_enable(False)
    fl = useful_flops(prob)
    rec = {"workload": WORKLOADS[workload]["desc"], "value": ms * 1e-3, "unit": "s", "ms_per_step": ms, "steps": steps, "warmup": warmup,
           "n": prob.n, "batch": prob.batch, "gpu_launches_per_step": int(launches), "useful_tflops": fl / (ms * 1e-3) / 1e12,
           "l2_policy": "inputs larger than L2" if flush is None else "L2 flushed between timed steps (256 MB write)",
           "phases_ms": {k: round(v, 3) for k, v in phases.items()}, "check": {"mu": mu},
           # which reduction the library took by itself: the band -> tridiagonal phase only exists on the two-stage path
           "reduction": "two_stage" if phases.get("band_to_tridiagonal", 0.0) > 0.02 * phases.get("tridiagonalise", 0.0)
                        else "one_stage"}
    if other_reduction:
        # the same step through the reduction the library did NOT pick (forced by flag): the measurement behind the default
        oflag = nao.NAO_TRD_ONE_STAGE if rec["reduction"] == "two_stage" else nao.NAO_TRD_TWO_STAGE
        try:
            owork = work
            need = nao.geneig_workspace(prob.n, prob.batch, dt, flags | oflag) + 256
            if need > work.numel():
                owork = torch.empty(need, dtype=torch.uint8, device=dev)

            def ostep():
                S.copy_(S0)
                E, C, info = nao.geneig(H, S, flags=flags | oflag, work=owork)
                mu_o, F = nao.fermi_mu(E, weights, prob.n_electrons, prob.kT)
                nao.density_matrix(C, F, out=Dbuf)
                return mu_o
            for _ in range(warmup):
                mu_o = ostep()
            torch.cuda.synchronize()
            tot = 0.0
            for _ in range(steps):
                if flush is not None:
                    flush.zero_()
                ev0.record(); ostep(); ev1.record(); torch.cuda.synchronize()
                tot += ev0.elapsed_time(ev1)
            rec["other_reduction"] = {"reduction": "one_stage" if oflag == nao.NAO_TRD_ONE_STAGE else "two_stage",
                                      "ms_per_step": tot / steps, "mu_difference": abs(mu_o - mu)}
            del owork
        except Exception as exc:
            rec["other_reduction"] = {"error": str(exc)}
    if cpu_certificate:
        try:
            rec["cpu_certificate"] = cpu_certificate_time(prob, last["E"], last["C"])
        except Exception as exc:
            rec["cpu_certificate"] = {"error": str(exc)}
    last.clear()
    if kp["launches"] > 0 and kp["ms"] > 0:
        ach = kp["work"] / (kp["ms"] * 1e-3) / 1e9
        tr, src = read_traffic("hetrd_panel_kernel", workload)
        rec["roofline"] = {"kernel": kp["name"], "bound": "hbm", "achieved": ach, "peak": hbm_peak, "unit": "GB/s", "frac": ach / hbm_peak,
                           "traffic": tr, "traffic_source": src, "kernel_ms_per_step": kp["ms"], "launches_per_step": kp["launches"],
                           "algorithmic_bytes_per_launch": kp["work"] / kp["launches"]}
    if kg["ms"] > 0:
        tf = kg["work"] / (kg["ms"] * 1e-3) / 1e12
        rec["roofline_gemm"] = {"kernel": kg["name"], "bound": "tensor", "achieved": tf, "peak": dmma_meas, "unit": "TFLOP/s",
                                "frac": tf / dmma_meas, "kernel_ms_per_step": kg["ms"], "launches_timed": kg["launches"]}
    # concurrent mid-size solves: the same step with the batch spread over 2/4/8 internal streams
    # (NAO_STREAM_GROUPS_*), against the single batched launch above
    if prob.batch >= 4 and groups:
        groups = {"1 (batched launches)": ms}
        for gname, gflag in (("2", nao.NAO_STREAM_GROUPS_2), ("4", nao.NAO_STREAM_GROUPS_4), ("8", nao.NAO_STREAM_GROUPS_8)):
            gwork = torch.empty(nao.geneig_workspace(prob.n, prob.batch, dt, flags | gflag) + 256, dtype=torch.uint8, device=dev)

            def gstep():
                S.copy_(S0)
                E, C, info = nao.geneig(H, S, flags=flags | gflag, work=gwork)
                mu, F = nao.fermi_mu(E, weights, prob.n_electrons, prob.kT)
                nao.density_matrix(C, F, out=Dbuf)
                return mu
            for _ in range(warmup):
                mu_g = gstep()
            torch.cuda.synchronize()
            assert abs(mu_g - mu) <= 1e-12
            tot = 0.0
            for _ in range(steps):
                if flush is not None:
                    flush.zero_()
                ev0.record(); gstep(); ev1.record(); torch.cuda.synchronize()
                tot += ev0.elapsed_time(ev1)
            groups[gname] = tot / steps
            del gwork
        rec["stream_groups_ms_per_step"] = groups
    del H, S, S0, work, Dbuf
    torch.cuda.empty_cache()
    return rec


def run_reference(args):
    """--impl reference: the CPU oracle timed on the host cores (rank 0 only)."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    vals = []
    for _ in range(args.warmup if args.warmup < 1 else 0):
        pass
    cb = None
    for _ in range(max(1, min(args.steps, 2))):
        cb = oracle_sample(args.workload)
        vals.append(cb["value"])
    v = sum(vals) / len(vals)
    cb["value"] = v
    line = {"impl": "reference", "metric": "s per SCF eigensolve+density matrix", "value": v, "unit": "s",
            "n_gpus": args.gpus, "steps": args.steps, "warmup": args.warmup, "ms_per_step": v * 1e3,
            "higher_is_better": False, "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": WORKLOADS[args.workload]["desc"], "parallelism": "host cores (oracle)"},
            "extrapolated": bool(cb.get("extrapolated")),
            "note": "the Jacobi oracle timed on a reduced-size replica of the workload and scaled by its N^3 law: context, "
                    "not a same-config measurement",
            "cpu_baseline": cb, "e2e": {"value": v, "unit": "s", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line))


def order_line(line):
    """Key order of the JSON line: the contract's scalars, then compact scalars of every config (a record that keeps only the
    head of the line still shows both halves of BASELINE.json's metric), then the contract's objects, then the long
    per-config sub-records."""
    def frac(rec, key):
        r = rec.get(key) if isinstance(rec, dict) else None
        return r.get("frac") if isinstance(r, dict) else None
    head = ["metric", "value", "unit", "n_gpus", "steps", "warmup", "ms_per_step", "higher_is_better", "scaling", "vs_baseline",
            "dtype", "data", "config", "gpu_launches", "reduction"]
    out = {k: line[k] for k in head if k in line}
    out["roofline_frac"] = frac(line, "roofline")
    if "roofline_hetrd" in line:
        out["hetrd_frac_one_stage_step"] = frac(line, "roofline_hetrd")
    if isinstance(line.get("e2e"), dict):
        out["e2e_ms_per_step"] = line["e2e"]["value"] * 1e3
    for wl in ("c3", "c1", "c4"):
        rec = line.get(wl)
        if isinstance(rec, dict) and "ms_per_step" in rec:
            out[wl + "_ms_per_step"] = rec["ms_per_step"]
            out[wl + "_hetrd_frac"] = frac(rec, "roofline")
            out[wl + "_gemm_frac"] = frac(rec, "roofline_gemm")
            out[wl + "_reduction"] = rec.get("reduction")
            if isinstance(rec.get("other_reduction"), dict) and "ms_per_step" in rec["other_reduction"]:
                out[wl + "_other_reduction_ms_per_step"] = rec["other_reduction"]["ms_per_step"]
    for k in ("roofline", "cpu_baseline", "e2e", "clocks", "roofline_hetrd", "roofline_gemm", "cpu_library", "cpu_oracle_c0"):
        if k in line:
            out[k] = line[k]
    for k, v in line.items():
        if k not in out:
            out[k] = v
    return out


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=5)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--workload", default="c2", choices=sorted(WORKLOADS))
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-side", action="store_true", help="skip the c3 / c1 / c4 side records of the default (c2) run")
    ap.add_argument("--reduction", default="default", choices=["default", "one_stage", "two_stage"],
                    help="force the tridiagonalisation path of the timed step (NAO_TRD_ONE_STAGE / NAO_TRD_TWO_STAGE)")
    ap.add_argument("--timed-only", action="store_true",
                    help="warm-up + timed steps only, minimal JSON line (the command the ncu launch lists are taken from)")
    args = ap.parse_args()
    if args.impl == "reference":
        return run_reference(args)

    import numpy as np
    import torch
    import paper_2606_09058_b200 as nao
    from paper_2606_09058_b200.synth import make_config

    rank = int(os.environ.get("RANK", "0")); world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: the product has no CPU path")
    torch.cuda.set_device(local)
    dev = torch.device("cuda", local)
    dist = None
    if world > 1:
        import torch.distributed as dist
        dist.init_process_group("nccl", device_id=dev)
    nao.lib()
    W = max(args.warmup, 3)

    from paper_2606_09058_b200.replicas import replica_seed
    prob = make_config(WORKLOADS[args.workload]["idx"], seed=replica_seed(rank))       # replicas: each rank its own seed
    flags = nao.NAO_NC_BLOCK_S if prob.nc_block_s else 0
    flags |= {"default": 0, "one_stage": nao.NAO_TRD_ONE_STAGE, "two_stage": nao.NAO_TRD_TWO_STAGE}[args.reduction]
    dt = nao.NAO_COMPLEX if prob.is_complex else nao.NAO_REAL
    # host (pinned) and device copies
    # the spin channels of a collinear Gamma-point calculation share one overlap matrix: it is passed once (strideS = 0)
    S_np = prob.S
    if not prob.nc_block_s and prob.S.shape[0] > 1 and all(np.array_equal(prob.S[0], prob.S[b]) for b in range(1, prob.S.shape[0])):
        S_np = np.ascontiguousarray(prob.S[:1])
    Hh = torch.from_numpy(prob.H).pin_memory(); Sh = torch.from_numpy(S_np).pin_memory()
    H = Hh.to(dev); S0 = Sh.to(dev); S = torch.empty_like(S0)
    work = torch.empty(nao.geneig_workspace(prob.n, prob.batch, dt, flags) + 256, dtype=torch.uint8, device=dev)
    Dbuf = torch.empty_like(H)
    Dh = torch.empty_like(Hh).pin_memory(); Eh = torch.empty((prob.batch, prob.n), dtype=torch.float64).pin_memory()
    weights = [float(x) for x in prob.weights]

    def step(f=flags, fresh_S=True):
        if fresh_S:
            S.copy_(S0)
        E, C, info = nao.geneig(H, S, flags=f, work=work)
        mu, F = nao.fermi_mu(E, weights, prob.n_electrons, prob.kT)
        D = nao.density_matrix(C, F, out=Dbuf)
        return E, C, info, mu, F, D

    def barrier():
        if dist is not None:
            dist.barrier()
        torch.cuda.synchronize()

    for _ in range(W):
        E, C, info, mu, F, D = step()
    torch.cuda.synchronize()
    assert int(info.abs().max()) == 0, "numerical failure: info=%s" % info.tolist()

    # ---- timed region: K full steps, device-resident inputs (708 MB of H at c2: larger than the 126 MB L2);
    #      no profiling events inside it
    sampler = ClockSampler(local); sampler.start()
    l0 = nao.launch_count()
    ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    in_bytes = H.numel() * H.element_size() + S0.numel() * S0.element_size()
    flush = None if in_bytes > (256 << 20) else torch.empty(256 << 20, dtype=torch.uint8, device=dev)
    barrier()
    if flush is None:
        ev0.record()
        for _ in range(args.steps):
            E, C, info, mu, F, D = step()
        ev1.record()
        barrier()
        ms = ev0.elapsed_time(ev1) / args.steps
    else:
        # small workloads: L2 (126 MB) is flushed by writing 256 MB between steps; every step has its own event pair
        tot = 0.0
        for _ in range(args.steps):
            flush.zero_()
            ev0.record()
            E, C, info, mu, F, D = step()
            ev1.record()
            torch.cuda.synchronize()
            tot += ev0.elapsed_time(ev1)
        barrier()
        ms = tot / args.steps
    launches = (nao.launch_count() - l0) // args.steps
    clocks = sampler.stop()
    if args.timed_only:
        if rank == 0:
            print(json.dumps({"metric": "s per SCF eigensolve+density matrix", "value": ms * 1e-3, "unit": "s", "ms_per_step": ms,
                              "steps": args.steps, "warmup": W, "timed_only": True, "reduction": args.reduction,
                              "config": {"workload": WORKLOADS[args.workload]["desc"]}, "gpu_launches": int(launches) * args.steps,
                              "clocks": clocks}))
        if dist is not None:
            dist.destroy_process_group()
        return

    # ---- one more step with the library's event timers on: phase boundaries and per-launch timers of the two
    #      kernel classes (slot 0 = hetrd_panel_kernel with its algorithmic HBM bytes, slot 1 = gemm_kernel with flops)
    nao.profile_enable(True)
    step()
    torch.cuda.synchronize()
    phases = nao.profile_read()
    kpanel = nao.profile_kernel(0)
    kgemm = nao.profile_kernel(1)
    nao.profile_enable(False)
    prof_steps = 1
    # which reduction the library's default took (real n >= 1536: two-stage; otherwise one-stage)
    default_path = "two_stage" if phases.get("band_to_tridiagonal", 0.0) > 0.05 else "one_stage"
    other_path = "one_stage" if default_path == "two_stage" else "two_stage"

    # ---- the same step through the OTHER reduction (one-stage HEMV-based / two-stage dense -> band -> tridiagonal)
    ms_two_stage, phases_two, kpanel_other = None, None, None
    big = work.numel() > (40 << 30)          # config 4: a second workspace does not fit next to the first one
    try:
        if big:
            raise RuntimeError("skipped: the comparison run needs a second workspace (> 40 GB)")
        f2 = flags | (nao.NAO_TRD_TWO_STAGE if other_path == "two_stage" else nao.NAO_TRD_ONE_STAGE)
        work2 = torch.empty(nao.geneig_workspace(prob.n, prob.batch, dt, f2) + 256, dtype=torch.uint8, device=dev)

        def step2():
            S.copy_(S0)
            E2, C2, info2 = nao.geneig(H, S, flags=f2, work=work2)
            mu2, F2 = nao.fermi_mu(E2, weights, prob.n_electrons, prob.kT)
            nao.density_matrix(C2, F2, out=Dbuf)
            return E2
        step2(); torch.cuda.synchronize()
        ev0.record()
        for _ in range(2):
            E2 = step2()
        ev1.record(); torch.cuda.synchronize()
        ms_two_stage = ev0.elapsed_time(ev1) / 2
        nao.profile_enable(True); step2(); torch.cuda.synchronize()
        phases_two = nao.profile_read(); kpanel_other = nao.profile_kernel(0); nao.profile_enable(False)
        assert float((E2 - E).abs().max()) <= 1e-9, "eigenvalues of the two reductions differ"
        del work2
    except Exception as exc:       # reported, never hidden
        phases_two = {"error": str(exc)}

    # ---- partial spectrum (nao_geneig_partial): only the eigenvectors the density matrix reads
    #      (f >= 1e-17, + 2 % margin) are back-transformed; same e, mu, D.  Reported beside the headline, which stays
    #      the full solve.
    partial = None
    try:
        if big:
            raise RuntimeError("skipped: the comparison run needs a second workspace (> 40 GB)")
        n_vec = min(prob.n, int(nao.occupied_count(F) * 1.02) + 8)
        res = {}
        for name, f3 in (("one_stage", flags | nao.NAO_S_FACTORED | nao.NAO_TRD_ONE_STAGE), ("two_stage", flags | nao.NAO_S_FACTORED | nao.NAO_TRD_TWO_STAGE)):
            w3 = torch.empty(nao.geneig_workspace(prob.n, prob.batch, dt, f3) + 256, dtype=torch.uint8, device=dev)

            def step3():
                E3, C3, info3 = nao.geneig(H, S, flags=f3, work=w3, n_vec=n_vec)
                mu3, F3 = nao.fermi_mu(E3, weights, prob.n_electrons, prob.kT)
                return nao.density_matrix(C3, F3, out=Dbuf), mu3
            Dref = D.clone()
            D3, mu3 = step3(); torch.cuda.synchronize()
            err = float((D3 - Dref).abs().max())
            ev0.record()
            for _ in range(2):
                step3()
            ev1.record(); torch.cuda.synchronize()
            res[name] = {"ms_per_step": ev0.elapsed_time(ev1) / 2, "max_abs_dD_vs_full": err, "dmu_vs_full": abs(mu3 - mu)}
            del w3, Dref
        partial = {"n_vec": n_vec, "n": prob.n, "step": "later SCF step (S factor cached)", **res}
    except Exception as exc:
        partial = {"error": str(exc)}

    # ---- fused call (nao_scf_step): the step takes the number of vectors from its own Fermi search and picks the reduction
    #      itself (two-stage from order 1536 on, real or complex)
    fused = None
    try:
        if big:
            raise RuntimeError("skipped: the comparison run needs a second workspace (> 40 GB)")
        res = {}
        for name, f4, fresh in (("first_step", flags, True), ("later_step", flags | nao.NAO_S_FACTORED, False)):
            def step4():
                if fresh:
                    S.copy_(S0)
                return nao.scf_step(H, S, weights, prob.n_electrons, prob.kT, flags=f4, out_D=Dbuf)
            Dref = D.clone()
            r4 = step4(); torch.cuda.synchronize()
            err = float((r4["D"] - Dref).abs().max())
            ev0.record()
            for _ in range(2):
                step4()
            ev1.record(); torch.cuda.synchronize()
            res[name] = {"ms_per_step": ev0.elapsed_time(ev1) / 2, "n_vec": r4["n_vec"], "max_abs_dD_vs_full": err,
                         "dmu_vs_full": abs(r4["mu"] - mu)}
            del Dref, r4
        fused = res
    except Exception as exc:
        fused = {"error": str(exc)}

    # later SCF steps reuse the factor of S: same path with NAO_S_FACTORED
    ev0.record()
    for _ in range(args.steps):
        step(flags | nao.NAO_S_FACTORED, fresh_S=False)
    ev1.record(); torch.cuda.synchronize()
    ms_later = ev0.elapsed_time(ev1) / args.steps

    # ---- end to end: host buffers in, host results out, every step
    #      (nao_solve_host: pinned host buffers through the C ABI; the library copies H on a second stream while S is
    #      factored and returns D item by item; the scratch of the device-resident run is released first)
    info_max = int(info.abs().max())
    # (the device-resident run's buffers are released first: at config 4 both sets do not fit side by side)
    del work, H, S, S0, Dbuf, E, C, F, D
    torch.cuda.empty_cache()
    need = ctypes.c_size_t(0)
    nao.lib().nao_solve_host_workspace(prob.n, prob.batch, dt, flags, 1 if Sh.shape[0] == 1 and prob.batch > 1 else 0, ctypes.byref(need))
    e2e_work = torch.empty(need.value + 256, dtype=torch.uint8, device=dev)

    def e2e_step():
        return nao.solve_host(Hh, Sh, weights, prob.n_electrons, prob.kT, flags=flags, device=dev, work=e2e_work, Eh=Eh, Dh=Dh)
    r_e2e = e2e_step(); barrier()
    assert abs(r_e2e["mu"] - mu) <= 1e-10 and int(r_e2e["info"].abs().max()) == 0
    ev0.record()
    for _ in range(args.steps):
        e2e_step()
    ev1.record(); barrier()
    ms_e2e = ev0.elapsed_time(ev1) / args.steps
    h2d = Hh.numel() * Hh.element_size() + Sh.numel() * Sh.element_size()
    d2h = Dh.numel() * Dh.element_size() + Eh.numel() * Eh.element_size()

    from paper_2606_09058_b200.replicas import max_over_ranks
    ms, ms_e2e, ms_later = max_over_ranks([ms, ms_e2e, ms_later], dist, dev)

    if rank == 0:
        peaks = {}
        try:
            peaks = json.load(open(os.path.join(ROOT, "MEASURED_PEAKS.json")))
        except Exception:
            pass
        hbm_peak = float(peaks.get("hbm_gbs", 6650.0))
        hbm_src = "measured (MEASURED_PEAKS.json hbm_gbs)" if "hbm_gbs" in peaks else "fallback 6.65 TB/s (B200_PROFILING.md)"
        # hetrd_panel_kernel (the HBM-bound BLAS2 tridiagonalisation) is timed in whichever of the two steps runs it
        hetrd_in_default = kpanel["launches"] > 0
        if not hetrd_in_default and kpanel_other is not None:
            kpanel = kpanel_other
        panel_ms = kpanel["ms"] / prof_steps
        panel_bytes = kpanel["work"] / prof_steps
        achieved = panel_bytes / (panel_ms * 1e-3) / 1e9 if panel_ms > 0 else 0.0
        fl = useful_flops(prob)
        gemm_tf = kgemm["work"] / (kgemm["ms"] * 1e-3) / 1e12 if kgemm["ms"] > 0 else 0.0
        dmma_meas = nao.dmma_peak()          # register-resident DMMA loop, measured in this run
        # DRAM traffic per launch from the committed ncu capture of this build (profiles/r02_traffic.csv)
        hetrd_wl = args.workload if hetrd_in_default else args.workload + "_one_stage"
        traffic, traffic_src = read_traffic("hetrd_panel_kernel", hetrd_wl)
        gemm_traffic, gemm_traffic_src = read_traffic("gemm_kernel", args.workload)
        line = {
            "metric": "s per SCF eigensolve+density matrix", "value": ms * 1e-3, "unit": "s", "n_gpus": world,
            "steps": args.steps, "warmup": W, "ms_per_step": ms, "higher_is_better": False, "scaling": "weak",
            "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": WORKLOADS[args.workload]["desc"], "n": prob.n, "batch": prob.batch,
                       "complex": bool(prob.is_complex), "parallelism": "replicas only (%d)" % world,
                       "l2_policy": ("inputs larger than L2 (H and S are %.0f MB)" % (in_bytes / 1e6)) if flush is None
                                    else "L2 flushed between timed steps (256 MB write)",
                       "step": "first SCF step: S factored inside the step",
                       "overlap": "one S shared by the items" if Sh.shape[0] == 1 and prob.batch > 1 else "one S per item"},
            "useful_tflops": fl / (ms * 1e-3) / 1e12, "useful_flops_per_step": fl,
            "fp64_dmma_peak_tflops": FP64_DMMA_PEAK_TFLOPS, "fp64_dmma_peak_measured_tflops": dmma_meas,
            "ms_per_step_later_scf_steps": ms_later,
            "phases_ms": {k: round(v, 3) for k, v in phases.items()},
            "reduction": default_path,
            "partial_spectrum": partial,
            "scf_step_fused": fused,
            other_path: {"ms_per_step": ms_two_stage, "note": "the same step through the other reduction (forced by flag)",
                         "phases_ms": phases_two and {k: round(v, 3) if isinstance(v, float) else v for k, v in phases_two.items()}},
            "e2e": {"value": ms_e2e * 1e-3, "unit": "s", "h2d_bytes_per_step": h2d, "d2h_bytes_per_step": d2h},
            "gpu_launches": int(launches) * args.steps,
            "clocks": clocks,
            "check": {"mu": mu, "info_max": info_max},
        }
        r_hetrd = {"kernel": kpanel["name"], "bound": "hbm", "achieved": achieved, "peak": hbm_peak, "unit": "GB/s",
                   "frac": achieved / hbm_peak if hbm_peak else None, "traffic": traffic, "traffic_source": traffic_src,
                   "peak_source": hbm_src, "kernel_ms_per_step": panel_ms, "launches_per_step": kpanel["launches"] // prof_steps,
                   "algorithmic_bytes_per_step": panel_bytes,
                   "algorithmic_bytes_per_launch": panel_bytes / max(1, kpanel["launches"] // prof_steps),
                   "measured_in": "the timed (default) step" if hetrd_in_default else "the one-stage comparison step"}
        r_gemm = {"kernel": kgemm["name"], "bound": "tensor", "achieved": gemm_tf, "peak": dmma_meas,
                  "unit": "TFLOP/s", "frac": gemm_tf / dmma_meas, "traffic": gemm_traffic, "traffic_source": gemm_traffic_src,
                  "peak_source": "measured in this run: register-resident DMMA.8x8x4 loop (nao_dmma_peak); derived "
                                 "148 SMs x 128 flop/clk x 1.965 GHz = 37.2; cuBLAS DGEMM reaches 35.6",
                  "kernel_ms_per_step": kgemm["ms"] / prof_steps, "launches_timed": kgemm["launches"],
                  "executed_flops_timed": kgemm["work"], "measured_in": "the timed (default) step"}
        # `roofline` = the kernel with the largest share of the timed step: hetrd_panel_kernel on the one-stage path,
        # the DMMA GEMM core (all its launches together) on the two-stage path; the other one is reported beside it
        if hetrd_in_default and panel_ms >= r_gemm["kernel_ms_per_step"]:
            line["roofline"], line["roofline_gemm"] = r_hetrd, r_gemm
        else:
            line["roofline"], line["roofline_hetrd"] = r_gemm, r_hetrd
        # the other headline workload of BASELINE.json's metric ("N=6656 real, 9984 cplx"), timed in the same run
        if world == 1 and args.workload == "c2" and not args.no_side:
            del e2e_work
            torch.cuda.empty_cache()
            for wl in ("c3", "c1", "c4"):
                try:
                    # config 4 (11.3 GB per matrix, 21 s per step): one warm-up and one timed step
                    kw = dict(steps=1, warmup=1) if wl == "c4" else {}
                    if wl == "c3" and not args.no_cpu_baseline:
                        kw["cpu_certificate"] = True
                    if wl in ("c3", "c1"):
                        kw["other_reduction"] = True
                    line[wl] = side_record(nao, torch, wl, dev, hbm_peak, dmma_meas, **kw)
                except Exception as exc:       # reported, never hidden
                    line[wl] = {"error": str(exc)}
        if not args.no_cpu_baseline and world == 1:
            line["cpu_baseline"] = oracle_sample(args.workload)
            try:
                line["cpu_library"] = cpu_library_time(args.workload)
            except Exception as exc:
                line["cpu_library"] = {"error": str(exc)}
            if args.workload == "c2" and not args.no_side:
                try:
                    inrun = oracle_in_run()
                    line["cpu_oracle_c0"] = inrun["c0"]
                    if isinstance(line.get("c1"), dict):
                        line["c1"]["cpu_oracle"] = inrun["c1"]
                except Exception as exc:
                    line["cpu_oracle_c0"] = {"error": str(exc)}
        print(json.dumps(order_line(line)))
    if dist is not None:
        dist.destroy_process_group()


if __name__ == "__main__":
    main()
