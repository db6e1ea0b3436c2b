"""tests/golden/c0_oracle.txt (written by tests/golden/make_golden.py from oracle/ only): the oracle must still reproduce it
(CPU), and the CUDA path must match it to the north_star tolerances (GPU)."""
import os

import numpy as np
import pytest

import oracle
from paper_2606_09058_b200.synth import make_config

GOLD = os.path.join(os.path.dirname(os.path.abspath(__file__)), "golden", "c0_oracle.txt")


def read_golden():
    g = {"e": {}, "D": {}}
    for line in open(GOLD):
        if line.startswith("#") or not line.strip():
            continue
        t = line.split()
        if t[0] == "e":
            g["e"][int(t[1])] = float(t[2])
        elif t[0] == "D":
            g["D"][(int(t[1]), int(t[2]))] = float(t[3])
        else:
            g[t[0]] = float(t[1])
    g["e"] = np.array([g["e"][k] for k in range(len(g["e"]))])
    return g


def test_oracle_reproduces_golden_config0():
    g = read_golden()
    prob = make_config(0)
    ref = oracle.solve_problem(prob)
    assert np.abs(ref["e"][0] - g["e"]).max() <= 1e-13
    assert abs(ref["mu"] - g["mu"]) <= 1e-13
    for (i, j), v in g["D"].items():
        assert abs(ref["D"][0][i, j] - v) <= 1e-13
    assert abs(g["trace_DS"] - prob.n_electrons / prob.weights[0]) <= 1e-10     # Tr(D S) = N_e / g


@pytest.mark.gpu
def test_cuda_path_matches_golden_config0():
    import torch
    import paper_2606_09058_b200 as nao
    g = read_golden()
    prob = make_config(0)
    dev = "cuda:0"
    E, C, info = nao.geneig(torch.from_numpy(prob.H).to(dev), torch.from_numpy(prob.S.copy()).to(dev))
    assert int(info.abs().max()) == 0
    mu, F = nao.fermi_mu(E, prob.weights, prob.n_electrons, prob.kT)
    D = np.swapaxes(nao.density_matrix(C, F).cpu().numpy(), -1, -2)[0]
    assert np.abs(E.cpu().numpy()[0] - g["e"]).max() <= 1e-9
    assert abs(mu - g["mu"]) <= 1e-10
    for (i, j), v in g["D"].items():
        assert abs(D[i, j] - v) <= 1e-8
    assert abs(np.linalg.norm(D) - g["norm_D_F"]) <= 1e-7
