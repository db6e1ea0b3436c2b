"""Writes tests/golden/c2_oracle.txt: the oracle's results for BASELINE config 2 (n = 6656 real, 2 spin channels sharing
one Fermi level, 2048 electrons, seed 0) from ONE full run of the Jacobi oracle ("at c2 once, offline,
stored as a small golden digest").

    OMP_NUM_THREADS=8 python tests/golden/make_golden_c2.py [--cache DIR]

Hours of CPU time (cyclic Jacobi, ~12 sweeps of n^3 long-double-accumulated work per item).  Calls only oracle/ and the
seeded input generator; never the CUDA path.  --cache keeps the per-item (e, C) so that an interrupted run resumes.
Stored (what is unique, reading of the gauge freedom): every eigenvalue of both items (Eq. 5), the
shared mu of the occupations f_i, diag(D), a seeded sample of entries of D = C diag(f) C^H (Eq. 8,
PAPER.md:63; reading C3), ||D||_F, Tr(D S), and a SHA-256 of the generator's output so a generator change is noticed."""
import argparse
import hashlib
import os
import sys
import time

import numpy as np

ROOT = os.path.dirname(os.path.dirname(os.path.dirname(os.path.abspath(__file__))))
sys.path.insert(0, ROOT)

import oracle  # noqa: E402
from paper_2606_09058_b200.synth import make_config  # noqa: E402

N_SAMPLES = 512


def sample_indices(n, count=N_SAMPLES, seed=20260609):
    """Seeded (i, j) pairs: numpy's PCG64 stream, fixed seed; independent of the method."""
    rng = np.random.Generator(np.random.PCG64(seed))
    return [(int(i), int(j)) for i, j in zip(rng.integers(0, n, count), rng.integers(0, n, count))]


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--cache", default=None)
    ap.add_argument("--nat", type=int, default=None, help="reduced-size dry run (writes c2_natN_oracle.txt)")
    args = ap.parse_args()
    prob = make_config(2, nat=args.nat)
    n = prob.n
    hh = hashlib.sha256()
    hh.update(np.ascontiguousarray(prob.H).tobytes())
    hh.update(np.ascontiguousarray(prob.S).tobytes())
    es, Cs, sweeps = [], [], []
    t_eig, t_den = 0.0, 0.0          # wall time of the oracle's eigensolves / density matrices of THIS run (cached items add 0)
    for b in range(prob.batch):
        cf = os.path.join(args.cache, "%s_item%d.npz" % (prob.name, b)) if args.cache else None
        if cf and os.path.exists(cf):
            z = np.load(cf)
            e, C, sw = z["e"], z["C"], int(z["sweeps"])
        else:
            t = time.time()
            e, C, info = oracle.geneig(prob.H_full(b), prob.S_full(b))
            sw = info["sweeps"]
            t_eig += time.time() - t
            print("item %d: %d sweeps, %.0f s" % (b, sw, time.time() - t), flush=True)
            if cf:
                os.makedirs(args.cache, exist_ok=True)
                np.savez(cf, e=e, C=C, sweeps=sw)
        es.append(e)
        Cs.append(C)
        sweeps.append(sw)
    e = np.stack(es)
    mu, f = oracle.fermi(e, prob.weights, prob.n_electrons, prob.kT)
    name = "c2_oracle.txt" if args.nat is None else "c2_nat%d_oracle.txt" % args.nat
    path = os.path.join(os.path.dirname(os.path.abspath(__file__)), name)
    samples = sample_indices(n)
    with open(path, "w") as fo:
        fo.write("# config 2 (BASELINE.json configs[2]): n=%d real, 2 spin items, g*w=1 each, %d electrons, kT=%.3e Ha, seed 0\n"
                 % (n, int(prob.n_electrons), prob.kT))
        fo.write("# written by tests/golden/make_golden_c2.py from oracle/ only (Cholesky reduction + cyclic Jacobi, long double);"
                 " Jacobi sweeps per item: %s\n" % sweeps)
        fo.write("generator_sha256 %s\n" % hh.hexdigest())
        fo.write("mu %.17e\n" % mu)
        for b in range(prob.batch):
            t = time.time()
            D = oracle.density(Cs[b], f[b])
            t_den += time.time() - t
            print("item %d: density %.0f s" % (b, time.time() - t), flush=True)
            fo.write("trace_DS %d %.17e\n" % (b, float(np.sum(D * prob.S_full(b).T))))
            fo.write("norm_D_F %d %.17e\n" % (b, float(np.linalg.norm(D))))
            for (i, j) in samples:
                fo.write("D %d %d %d %.17e\n" % (b, i, j, D[i, j]))
            for k in range(n):
                fo.write("diagD %d %d %.17e\n" % (b, k, D[k, k]))
            for k in range(n):
                fo.write("e %d %d %.17e\n" % (b, k, e[b, k]))
    # wall times of this run, read by bench.py (cpu_baseline.full_run, tagged "recorded": a record of this script's run, not a
    # measurement of the bench run)
    import json
    with open(path[:-4] + "_run.json", "w") as fo:
        json.dump({"recorded": True, "eigensolve_s": round(t_eig), "density_s": round(t_den),
                   "threads": int(os.environ.get("OMP_NUM_THREADS", os.cpu_count() or 1)), "host_cores": os.cpu_count(),
                   "sweeps": sweeps, "source": "tests/golden/make_golden_c2.py"}, fo, indent=1)
        fo.write("\n")
    print(path)


if __name__ == "__main__":
    main()
