"""CPU-only checks of the boundary: the C-ABI library builds for sm_100a, loads without a GPU
and exports every function include/ants_recon.h declares; the binding fails loudly (no fallback)
when there is no CUDA device.  No compute calls here."""
import ctypes
import os
import re
import subprocess

import numpy as np
import pytest

from paper_1602_07247_b200 import build, recon, synth

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
HEADER = os.path.join(ROOT, "include", "ants_recon.h")


def declared_functions():
    src = open(HEADER).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(ants_[a-z0-9_]+)\s*\(", src)))


def test_header_declares_the_north_star_calls():
    names = declared_functions()
    for n in ("ants_lrf_create", "ants_reconstruct", "ants_destroy"):
        assert n in names


def test_library_builds_loads_and_exports_every_declared_symbol():
    path = build.build()
    assert os.path.exists(path)
    lib = ctypes.CDLL(path)
    for name in declared_functions():
        assert hasattr(lib, name), name
    # the object really is sm_100a device code
    out = subprocess.run(["cuobjdump", "-lelf", path], capture_output=True, text=True)
    if out.returncode == 0:
        assert "sm_100a" in out.stdout


def test_header_is_plain_c():
    """The boundary has no C++/torch types: the header compiles as C99."""
    r = subprocess.run(["gcc", "-std=c99", "-fsyntax-only", "-x", "c", HEADER], capture_output=True, text=True)
    assert r.returncode == 0, r.stderr


def test_strerror_and_struct_layout():
    recon.load()
    assert recon.strerror(0) == "ok"
    assert "invalid" in recon.strerror(-1)
    assert ctypes.sizeof(recon.LrfDims) == 20 and ctypes.sizeof(recon.GridParams) == 32


def test_no_cpu_fallback_without_a_gpu():
    import torch
    if torch.cuda.is_available():
        pytest.skip("has a GPU")
    cfg = synth.make_config(1)
    with pytest.raises(recon.AntsError) as ei:
        recon.Reconstructor(cfg)
    assert ei.value.status == -3          # ANTS_ERR_CUDA: no device, nothing is computed on the host


def test_invalid_model_arguments_are_rejected_before_any_gpu_work():
    cfg = synth.make_config(1)
    bad = [
        dict(knots=np.array([5.0, 1.0], np.float32)),                     # unordered knots
        dict(knots=np.array([0.0, np.inf], np.float32)),
        dict(dims=recon.LrfDims(cfg.n_sensors, 3, 1, 16, 0)),             # n_lrf neither 1 nor N
        dict(dims=recon.LrfDims(0, 1, 1, 16, 0)),
        dict(dims=recon.LrfDims(cfg.n_sensors, 1, 3, 16, 0)),
        dict(gains=np.zeros(cfg.n_sensors, np.float32)),
    ]
    for kw in bad:
        a = dict(sensor_xy=cfg.sensor_xy, gains=cfg.gains, knots=cfg.knots, coeffs=cfg.coeffs,
                 dims=recon.LrfDims(cfg.n_sensors, 1, 1, 16, 0))
        a.update(kw)
        with pytest.raises(recon.AntsError) as ei:
            recon.ants_lrf_create(a["sensor_xy"], a["gains"], a["knots"], a["coeffs"], a["dims"])
        assert ei.value.status == -1, kw


def test_distance_grouping_in_the_library_agrees_with_the_oracle():
    """ants_group_by_radius is host-only: it runs without a GPU.  The oracle's grouping (oracle/fit.py, pinned by
    hex ring counts in tests/test_oracle_fit.py) is the reference."""
    from oracle import fit as ofit
    for xy in (synth.hex_array(1, 30.0), synth.hex_array(3, 30.0), synth.hex_array(6, 25.0), synth.square_array(8, 6.0)):
        g, n = recon.ants_group_by_radius(xy)
        g0, n0 = ofit.group_by_radius(xy)
        assert n == n0 and np.array_equal(g, g0)
    with pytest.raises(recon.AntsError):
        recon.ants_group_by_radius(synth.hex_array(1, 30.0), tol=-1.0)


def test_gain_renormalisation_in_the_library_agrees_with_the_oracle():
    from oracle import fit as ofit
    rng = np.random.default_rng(5)
    prev = rng.uniform(0.5, 1.5, 37).astype(np.float32)
    new = (prev * rng.uniform(0.9, 1.1, 37) * 3.7).astype(np.float32)
    new[[3, 11]] = np.nan
    new[20] = -0.25
    out = recon.ants_gains_renormalise(new, prev)
    ref = ofit.renormalise_gains(new, prev)
    assert np.array_equal(out, ref)
    bad = prev.copy()
    bad[0] = 0.0
    with pytest.raises(recon.AntsError):
        recon.ants_gains_renormalise(new, bad)
