"""Per-kernel measurement entry of libnao.so building blocks (CUDA events, warm-up, L2 flush between repetitions): the
command the ncu captures summarised under profiles/ run.  Library kernels only.

    python -m paper_2606_09058_b200.microbench gemm [--m M --n N --k K] [--complex] [--opa 0|1|2] [--opb 0|1|2]
                                                    [--beta B] [--lower] [--reps R]
    python -m paper_2606_09058_b200.microbench heev [--n N] [--batch B] [--complex] [--two-stage|--one-stage]
    python -m paper_2606_09058_b200.microbench fold [--n N] [--nk NK] [--nr NR] [--complex]      (config 1: 832, 8, 27)
    python -m paper_2606_09058_b200.microbench fermi [--n N] [--batch B]                         (config 2: 6656, 2; config 1: 832, 16)

Prints one JSON line per measurement.
"""
from __future__ import annotations

import argparse
import json

import torch

from . import binding as B

FP64_DMMA_PEAK_TFLOPS = 148 * 128 * 1.965e9 / 1e12


def _flush_l2(buf):
    buf.zero_()


def _time(fn, reps, flush):
    ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    for _ in range(3):
        fn()
    times = []
    for _ in range(reps):
        _flush_l2(flush)
        ev0.record()
        fn()
        ev1.record()
        torch.cuda.synchronize()
        times.append(ev0.elapsed_time(ev1))
    times.sort()
    return times[len(times) // 2]


def bench_gemm(args):
    dev = torch.device("cuda:0")
    m, n, k = args.m, args.n, args.k
    dt = torch.complex128 if args.complex else torch.float64
    g = torch.Generator(device=dev)
    g.manual_seed(0)

    def rnd(cols, rows):
        x = torch.randn(1, cols, rows, dtype=torch.float64, device=dev, generator=g)
        if args.complex:
            x = torch.complex(x, torch.randn(1, cols, rows, dtype=torch.float64, device=dev, generator=g))
        return x

    # column-major items: shape (batch, cols, rows)
    A = rnd(k, m) if args.opa == 0 else rnd(m, k)
    Bm = rnd(n, k) if args.opb == 0 else rnd(k, n)
    C = torch.zeros(1, n, m, dtype=dt, device=dev)
    flush = torch.empty(256 << 20, dtype=torch.uint8, device=dev)
    ms = _time(lambda: B.gemm(A, Bm, args.opa, args.opb, 1.0, args.beta, C=C, lower_only=args.lower), args.reps, flush)
    flops = (8.0 if args.complex else 2.0) * m * n * k * (0.5 if args.lower else 1.0)
    out = {"kernel": "gemm_kernel", "m": m, "n": n, "k": k, "complex": args.complex, "opA": args.opa, "opB": args.opb,
           "beta": args.beta, "lower_only": args.lower, "ms": ms, "tflops": flops / ms / 1e9,
           "frac_of_dmma_peak": flops / ms / 1e9 / FP64_DMMA_PEAK_TFLOPS}
    print(json.dumps(out))


def bench_heev(args):
    dev = torch.device("cuda:0")
    n, batch = args.n, args.batch
    g = torch.Generator(device=dev)
    g.manual_seed(1)
    A = torch.randn(batch, n, n, dtype=torch.float64, device=dev, generator=g)
    if args.complex:
        A = torch.complex(A, torch.randn(batch, n, n, dtype=torch.float64, device=dev, generator=g))
    A = A + A.mH
    flags = B.NAO_TRD_TWO_STAGE if args.two_stage else (B.NAO_TRD_ONE_STAGE if args.one_stage else 0)
    res = {}
    for it in range(max(2, args.reps)):
        B.profile_enable(True)
        E, Z, info = B.heev(A.clone(), flags=flags)
        torch.cuda.synchronize()
        res = B.profile_read()
        kp = [B.profile_kernel(s) for s in range(2)]
        B.profile_enable(False)
    Zm = Z[0].T                                     # column-major item -> logical matrix
    Am = A[0].T
    r = (Am @ Zm - Zm * E[0][None, :]).abs().max().item()
    o = (Zm.mH @ Zm - torch.eye(n, dtype=Zm.dtype, device=dev)).abs().max().item()
    print(json.dumps({"kernel": "heev", "n": n, "batch": batch, "complex": args.complex, "flags": flags,
                      "phases_ms": {k: round(v, 3) for k, v in res.items()}, "kernels": kp,
                      "residual_max": r, "orth_max": o, "info": info.tolist()}))


def bench_fold(args):
    """nao_fold_density: D(R) = sum_k w_k exp(-i k.R) D(k); HBM-bound (every D(k) element read once, every D(R) element
    written once).  --complex writes complex D(R), default is the real part only."""
    dev = torch.device("cuda:0")
    g = torch.Generator(device=dev)
    g.manual_seed(0)
    n, nk, nR = args.n, args.nk, args.nr
    Dk = torch.complex(torch.randn(nk, n, n, dtype=torch.float64, device=dev, generator=g),
                       torch.randn(nk, n, n, dtype=torch.float64, device=dev, generator=g))
    L = 10.8
    kp = [[6.283185307179586 * 0.25 * (1 if (q >> d) & 1 else -1) / L * (1 + q // 8) for d in range(3)] for q in range(nk)]
    w = [1.0 / nk] * nk
    Rv = [[L * ((r // 9) % 3 - 1), L * ((r // 3) % 3 - 1), L * (r % 3 - 1 + 3 * (r // 27))] for r in range(nR)]
    flush = torch.empty(256 << 20, dtype=torch.uint8, device=dev)
    ms = _time(lambda: B.fold_density(Dk, kp, w, Rv, real_out=not args.complex), args.reps, flush)
    by = n * n * (16.0 * nk + (16.0 if args.complex else 8.0) * nR)
    print(json.dumps({"kernel": "fold_density", "n": n, "nk": nk, "nR": nR, "complex_out": bool(args.complex), "ms": ms,
                      "algorithmic_bytes": by, "GBps": by / ms / 1e6}))


def bench_fermi(args):
    """nao_fermi_mu (rank sort + single-CTA bisection + occupations; the call synchronises the stream) and its workspace-free
    twin on a seeded spectrum with a gap at the filling (plain form of the search) and at exact integer filling of a gapped
    spectrum (log form): n levels per item in [-3, 3] Ha with the levels between -0.05 and 0.05 removed, kT = 9.5e-4 Ha."""
    n, batch = args.n, args.batch
    g = torch.Generator(device="cuda"); g.manual_seed(7)
    E = torch.rand((batch, n), dtype=torch.float64, device="cuda", generator=g) * 2.95 + 0.05
    E[:, : n // 3] *= -1.0
    E = torch.sort(E, dim=1).values.contiguous()
    w = [2.0 / batch] * batch
    flush = torch.empty(256 << 20, dtype=torch.uint8, device="cuda")
    for name, ne in (("plain", 2.0 * (n // 3) - 0.37), ("log", 2.0 * (n // 3))):
        mu = [0.0]

        def run():
            mu[0], _ = B.fermi_mu(E, w, ne, 9.5e-4)
        ms = _time(run, args.reps, flush)
        mu_static = None
        if n * batch <= B.FERMI_STATIC_MAX_STATES:
            mu_static, _ = B.fermi_mu_static(E, w, ne, 9.5e-4)
        print(json.dumps({"kernel": "nao_fermi_mu", "form": name, "n": n, "batch": batch, "states": n * batch, "ms": ms,
                          "mu": mu[0], "mu_static_minus_mu": None if mu_static is None else mu_static - mu[0]}))


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("what", choices=["gemm", "heev", "fold", "fermi"])
    ap.add_argument("--nk", type=int, default=8)
    ap.add_argument("--nr", type=int, default=27)
    ap.add_argument("--m", type=int, default=6656)
    ap.add_argument("--n", type=int, default=6656)
    ap.add_argument("--k", type=int, default=6656)
    ap.add_argument("--batch", type=int, default=1)
    ap.add_argument("--complex", action="store_true")
    ap.add_argument("--opa", type=int, default=0)
    ap.add_argument("--opb", type=int, default=0)
    ap.add_argument("--beta", type=float, default=0.0)
    ap.add_argument("--lower", action="store_true")
    ap.add_argument("--two-stage", action="store_true")
    ap.add_argument("--one-stage", action="store_true")
    ap.add_argument("--reps", type=int, default=5)
    args = ap.parse_args()
    if not torch.cuda.is_available():
        raise SystemExit("microbench needs a CUDA device: the product has no CPU path")
    B.lib()
    {"gemm": bench_gemm, "heev": bench_heev, "fold": bench_fold, "fermi": bench_fermi}[args.what](args)


if __name__ == "__main__":
    main()
