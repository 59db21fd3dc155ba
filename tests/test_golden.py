"""Stored expected values (tests/golden/*.txt, written by tests/golden/make_golden.py from oracle/ only).

CPU: the oracle and the seeded generators still reproduce them (a change to either is then a deliberate, reviewed
regeneration).  GPU: the CUDA path reproduces them through the C-ABI (fp64 D_w to 1e-13 relative to the field norm,
the solve to the solve tolerance) -- a check that does not need the oracle at run time.
"""
import importlib.util
import os

import numpy as np
import pytest

HERE = os.path.dirname(os.path.abspath(__file__))
spec = importlib.util.spec_from_file_location("make_golden", os.path.join(HERE, "golden", "make_golden.py"))
mg = importlib.util.module_from_spec(spec)
spec.loader.exec_module(mg)


def read_golden(case):
    out = {}
    with open(os.path.join(HERE, "golden", f"{case}.txt")) as f:
        for line in f:
            if line.startswith("#"):
                continue
            c, name, i, re, im = line.split()
            assert c == case
            out.setdefault(name, []).append((int(i), complex(float(re), float(im))))
    return out


@pytest.mark.parametrize("case", list(mg.CASES))
def test_oracle_reproduces_golden(case):
    gold = read_golden(case)
    q = mg.quantities(case)
    assert set(gold) == set(q)
    for name, rows in gold.items():
        scale = np.max(np.abs(q[name]))
        tol = {"eta": 0.0, "Dw_eta": 1e-14, "solve": 1e-11}[name]   # solve: CG to 1e-13, cond(D) ~ 10
        for i, z in rows:
            assert abs(q[name][i] - z) <= tol * scale, (name, i)


@pytest.mark.gpu
@pytest.mark.parametrize("case", list(mg.CASES))
def test_cuda_reproduces_golden(case):
    import synth
    from paper_2502_02490_b200 import binding as B
    c = mg.CASES[case]
    gold = read_golden(case)
    g = B.Qxd(*c["dims"], c["cstar"] | (c["ap"] << 2), precisions=(B.QXD_F64,))
    U = synth.su3_links(c["dims"], c["eps"], 1)
    A = synth.u1_field(c["dims"], 0.3, 2) if c["qed"] else None
    g.gauge_load(U, A, 1.0)
    g.set_quark(c["kappa"], c["q"])
    g.clover_build(c["csw"], c["csw_qed"])
    eta = synth.gaussian_spinor(g.dims_ext, 3)
    for i, z in gold["eta"]:
        assert eta.ravel()[i] == z
    dw = g.apply_Dw(eta, B.QXD_F64).cpu().numpy().ravel()
    scale = max(abs(z) for _, z in gold["Dw_eta"])
    for i, z in gold["Dw_eta"]:
        assert abs(dw[i] - z) <= 1e-13 * scale
    psi, info = g.solve(eta, 1e-12, algo=B.QXD_CGNE, sloppy=B.QXD_F64)
    assert info["status"] == 0
    psi = psi.cpu().numpy().ravel()
    scale = max(abs(z) for _, z in gold["solve"])
    for i, z in gold["solve"]:
        assert abs(psi[i] - z) <= 1e-10 * scale
    g.close()
