"""Writes tests/golden/*.txt from the fp64 CPU oracle ONLY (never from the CUDA path).

    python tests/golden/make_golden.py

The paper (arxiv 2502.02490) prints no operator values, so these files are not paper fixtures: they freeze what
the pinned oracle (tests/test_oracle_pins.py) computes for BASELINE.json configs c0 and a half-size c1, so that a
later change to the oracle's arithmetic, to synth/ (the seeded inputs) or to the site order at the ABI boundary
(Eq. (1)) is noticed.  Format per line: case, quantity, flat index, real part, imaginary part (%.17e).
"""
import os
import sys

import numpy as np

HERE = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, os.path.dirname(os.path.dirname(HERE)))
import synth  # noqa: E402
from oracle import qxd_ref as R  # noqa: E402

CASES = {
    # BASELINE.json configs[0]: 4x4^3 QCD, antiperiodic in time, kappa 0.12, csw 1.5, eps 0.3, seed 1
    "c0": dict(dims=(4, 4, 4, 4), cstar=0, ap=1, qed=False, q=0.0, kappa=0.12, csw=1.5, csw_qed=0.0, eps=0.3),
    # BASELINE.json configs[1] at half the extent (4x4^3 physical, doubled in x1): C* in 3 directions, QCD+QED, q = -1/3
    "c1h": dict(dims=(4, 4, 4, 4), cstar=3, ap=1, qed=True, q=-1.0 / 3.0, kappa=0.12, csw=1.5, csw_qed=1.0, eps=0.3),
}
NSAMPLE = 24


def build(case):
    c = CASES[case]
    ref = R.Ref(*c["dims"], c["cstar"] | (c["ap"] << 2))
    U = synth.su3_links(c["dims"], c["eps"], 1)
    A = synth.u1_field(c["dims"], 0.3, 2) if c["qed"] else None
    ref.gauge_load(U, A, 1.0)
    ref.set_quark(c["kappa"], c["q"])
    ref.clover_build(c["csw"], c["csw_qed"])
    eta = synth.gaussian_spinor(ref.dims_ext, 3)
    return ref, eta


def sample_indices(n):
    # fixed, spread over the whole field (first, last, and a stride coprime to every extent)
    idx = sorted(set([0, n - 1] + [(k * 7919 + 13) % n for k in range(NSAMPLE - 2)]))
    return idx


def quantities(case):
    ref, eta = build(case)
    out = {"eta": eta.ravel(), "Dw_eta": ref.apply_Dw(eta).ravel()}
    psi, _ = ref.solve(eta, 1e-13)
    out["solve"] = np.asarray(psi).ravel()
    return out


def main():
    for case in CASES:
        q = quantities(case)
        path = os.path.join(HERE, f"{case}.txt")
        with open(path, "w") as f:
            f.write(f"# written by tests/golden/make_golden.py from oracle/ only; case {case}: {CASES[case]}\n")
            for name, v in q.items():
                for i in sample_indices(v.size):
                    f.write(f"{case} {name} {i} {v[i].real:.17e} {v[i].imag:.17e}\n")
        print("wrote", path)


if __name__ == "__main__":
    main()
