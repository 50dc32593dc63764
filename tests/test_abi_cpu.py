"""CPU-side checks of the boundary: the library builds, loads and exports every symbol include/rift_ile.h declares;
argument validation that needs no GPU; the binding fails loudly when the library is missing."""
import os
import re

import numpy as np
import pytest

import paper_2210_07912_b200 as pkg
from paper_2210_07912_b200 import binding, build as build_mod

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def test_library_builds_and_exports_every_declared_symbol():
    path = build_mod.build()
    assert os.path.exists(path)
    header = open(os.path.join(ROOT, "include", "rift_ile.h")).read()
    declared = set(re.findall(r"\b(rift_ile_[a-z_]+)\s*\(", header))
    declared.discard("rift_ile_t")
    assert declared == set(binding.EXPORTS), declared ^ set(binding.EXPORTS)
    L = binding.lib()
    for name in declared:
        assert hasattr(L, name), name
    header_ac = open(os.path.join(ROOT, "include", "rift_ac.h")).read()
    declared_ac = set(re.findall(r"\b(rift_ac_[a-z_]+)\s*\(", header_ac))
    assert declared_ac == set(binding.AC_EXPORTS), declared_ac ^ set(binding.AC_EXPORTS)
    for name in declared_ac:
        assert hasattr(L, name), name
    header_sky = open(os.path.join(ROOT, "include", "rift_sky.h")).read()
    declared_sky = set(re.findall(r"\b(rift_sky_[a-z_]+)\s*\(", header_sky))
    assert declared_sky == set(binding.SKY_EXPORTS), declared_sky ^ set(binding.SKY_EXPORTS)
    for name in declared_sky:
        assert hasattr(L, name), name
    header_gmm = open(os.path.join(ROOT, "include", "rift_gmm.h")).read()
    declared_gmm = set(re.findall(r"\b(rift_gmm_[a-z_]+)\s*\(", header_gmm))
    assert declared_gmm == set(binding.GMM_EXPORTS), declared_gmm ^ set(binding.GMM_EXPORTS)
    for name in declared_gmm:
        assert hasattr(L, name), name
    # the frame is host arithmetic: checked here against its definition (pole = baseline, right-handed, x' equatorial)
    R = binding.rift_sky_network_frame([1.0, 2.0, 3.0], [4.0, 0.0, 5.0])
    z = np.array([3.0, -2.0, 2.0]) / np.sqrt(17.0)
    assert np.allclose(R[:, 2], z) and np.allclose(R.T @ R, np.eye(3)) and abs(np.linalg.det(R) - 1) < 1e-14 and R[2, 0] == 0.0
    with pytest.raises(binding.RiftError):
        binding.rift_sky_network_frame([1.0, 2.0, 3.0], [1.0, 2.0, 3.0])


def test_strerror_and_invalid_arguments_without_gpu():
    assert pkg.rift_ile_strerror(0) == "ok"
    assert "window" in pkg.rift_ile_strerror(pkg.RIFT_EWINDOW)
    loc = np.array([[6.3e6, 0, 0], [0, 6.3e6, 0]])
    resp = np.zeros((2, 3, 3))
    z = lambda *s: np.zeros(s, dtype=complex)
    mk = lambda **kw: pkg.rift_ile_create(**{**dict(det_location_m=loc, det_response=resp, gmst_rad=0.0, mode_l=[2, 2],
                                                    mode_m=[2, -2], n_points=1, n_t=411, delta_t=1 / 4096, n_tau=411,
                                                    d_ref_mpc=1000.0, Q=z(1, 2, 2, 411), U=z(1, 2, 2, 2),
                                                    V=z(1, 2, 2, 2)), **kw})
    for bad in (dict(mode_l=[2, 2], mode_m=[2, 2]), dict(mode_l=[1, 2]), dict(mode_m=[3, 2]), dict(n_tau=410),
                dict(n_tau=413), dict(delta_t=0.0), dict(d_ref_mpc=-1.0), dict(n_points=0),
                dict(precision=pkg.RIFT_PREC_FP64, q_storage=pkg.RIFT_Q_C64)):
        with pytest.raises(pkg.RiftError) as e:
            mk(**bad)
        assert e.value.code == pkg.RIFT_EINVAL, bad
    # guard band: S_max = ceil(6.3e6 / c / dt) = 87 samples -> n_tau + 174 must fit in n_t
    with pytest.raises(pkg.RiftError) as e:
        mk(n_tau=411 - 2 * 80)
    assert e.value.code == pkg.RIFT_EWINDOW


def test_missing_library_fails_loudly(monkeypatch, tmp_path):
    monkeypatch.setattr(binding, "_lib", None)
    monkeypatch.setattr(binding, "LIB_PATH", str(tmp_path / "nope.so"))
    with pytest.raises(ImportError):
        binding.lib()


def test_product_does_not_import_the_oracle():
    for dirpath, _d, files in os.walk(os.path.join(ROOT, "paper_2210_07912_b200")):
        for f in files:
            if f.endswith((".py", ".cu", ".h", ".cuh")):
                src = open(os.path.join(dirpath, f)).read()
                assert "import oracle" not in src and "from oracle" not in src and "liboracle" not in src, f
    for f in os.listdir(os.path.join(ROOT, "oracle")):
        if f.endswith((".py", ".c")):
            src = open(os.path.join(ROOT, "oracle", f)).read()
            assert "import paper_2210_07912_b200" not in src and "from paper_2210_07912_b200" not in src, f
