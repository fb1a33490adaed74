"""Seeded input generator (paper_2111_04457_b200/inputs): SU(3)-ness, determinism, distribution.  CPU only."""
import os
import subprocess
import sys

import numpy as np

from paper_2111_04457_b200 import inputs


def test_links_are_su3():
    for eps in (0.3, 0.5, 0.7):
        U = inputs.gauge((4, 4, 4, 6), 123, eps)
        UUd = np.einsum("...ij,...kj->...ik", U, U.conj())
        assert np.abs(UUd - np.eye(3)).max() < 1e-14
        assert np.abs(np.linalg.det(U) - 1).max() < 1e-14
        # roughness grows with eps: mean Re tr U / 3 decreases
    tr = [np.trace(inputs.gauge((4, 4, 4, 4), 1, e), axis1=-2, axis2=-1).real.mean() / 3 for e in (0.3, 0.5, 0.7)]
    assert tr[0] > tr[1] > tr[2] > 0


def test_links_match_expm_of_hermitian():
    """exp(i eps H) with H traceless Hermitian: eigenvalue phases of U sum to 0 and U(eps)^2 = U(2 eps)."""
    U1 = inputs.gauge((2, 2, 2, 2), 9, 0.25)
    U2 = inputs.gauge((2, 2, 2, 2), 9, 0.5)
    assert np.abs(U1 @ U1 - U2).max() < 1e-13


def test_source_is_unit_complex_gaussian():
    psi = inputs.spinor((8, 8, 8, 8), 42)
    assert abs(psi.real.mean()) < 0.01 and abs(psi.imag.mean()) < 0.01
    assert abs(psi.real.var() - 1) < 0.02 and abs(psi.imag.var() - 1) < 0.02
    assert abs(np.mean(psi.real * psi.imag)) < 0.01


def test_deterministic_and_stream_separated():
    a = inputs.spinor((4, 4, 4, 4), 7)
    assert np.array_equal(a, inputs.spinor((4, 4, 4, 4), 7))
    assert not np.array_equal(a, inputs.spinor((4, 4, 4, 4), 8))
    assert not np.array_equal(a, inputs.spinor((4, 4, 4, 4), 7, inputs.STREAM_TEST))
    # counter based: a smaller lattice is a prefix of the stream
    assert np.array_equal(inputs.spinor((4, 4, 4, 2), 7).ravel(), a.ravel()[: 12 * 128])


def test_independent_of_thread_count():
    code = ("import numpy as np, hashlib; from paper_2111_04457_b200 import inputs;"
            "print(hashlib.sha256(inputs.gauge((4,4,4,4), 3, 0.3).tobytes()).hexdigest())")
    root = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
    outs = []
    for nt in ("1", "4"):
        env = dict(os.environ, OMP_NUM_THREADS=nt, PYTHONPATH=root)
        outs.append(subprocess.run([sys.executable, "-c", code], env=env, capture_output=True, text=True,
                                   check=True).stdout.strip())
    assert outs[0] == outs[1]


def test_golden_config1():
    """Drift guard (tests/golden/README.md): the seeded inputs and the oracle reproduce the stored numbers of config 1."""
    import importlib.util
    import json
    import os
    here = os.path.join(os.path.dirname(os.path.abspath(__file__)), "golden")
    spec = importlib.util.spec_from_file_location("make_golden", os.path.join(here, "make_golden.py"))
    mod = importlib.util.module_from_spec(spec)
    spec.loader.exec_module(mod)
    now = mod.compute()
    with open(os.path.join(here, "config1_oracle.json")) as f:
        ref = json.load(f)
    assert set(now) == set(ref)
    for k, v in ref.items():
        if k.startswith("_"):
            continue
        if k.startswith("bicgstab_iters"):
            assert abs(now[k] - v) <= 2, k
        else:
            assert np.allclose(now[k], v, rtol=1e-11, atol=1e-11), (k, now[k], v)
