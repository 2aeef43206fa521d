"""CPU-only checks of the C ABI: the library loads, exports every symbol the
header declares, validates descriptors, and its host-side logic (sample
count, slab plan) agrees with the oracle / hand arithmetic.  No compute calls."""
import os
import re

import numpy as np
import pytest

from paper_2512_21180_b200 import synth

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def cbct():
    from paper_2512_21180_b200 import build, cbct as m
    build.build()
    m.load_library()
    return m


def test_exports_match_header(cbct):
    hdr = open(os.path.join(ROOT, "include", "cbct.h")).read()
    declared = set(re.findall(r"\b(cbct_[a-z_]+)\s*\(", hdr))
    assert declared == set(cbct.EXPORTS), declared ^ set(cbct.EXPORTS)
    lib = cbct.load_library()
    for name in declared:
        assert getattr(lib, name) is not None


def test_static_scratch_limit_matches_header(cbct):
    """The binding's STATIC_SCRATCH_BYTES is the header's CBCT_STATIC_SCRATCH_BYTES (cbct_bp_fdk_static)."""
    hdr = open(os.path.join(ROOT, "include", "cbct.h")).read()
    m = re.search(r"#define\s+CBCT_STATIC_SCRATCH_BYTES\s+\((\d+)u\s*<<\s*(\d+)\)", hdr)
    assert m, "CBCT_STATIC_SCRATCH_BYTES not found in include/cbct.h"
    assert int(m.group(1)) << int(m.group(2)) == cbct.STATIC_SCRATCH_BYTES


def test_status_strings(cbct):
    lib = cbct.load_library()
    assert lib.cbct_status_string(0) == b"CBCT_OK"
    for rc in (-1, -2, -3, -4):
        assert lib.cbct_status_string(rc).startswith(b"CBCT_ERR")


@pytest.mark.parametrize("bad", [
    dict(step_vox=0.0), dict(step_vox=1.5), dict(n_views=0), dict(det_nu=0), dict(vox_mm=-1.0),
    dict(sdd_mm=900.0), dict(vol_nx=500, vox_mm=4.0),  # volume reaches the source orbit
    dict(vol_cx_mm=float("nan")),
])
def test_create_rejects_bad_geometry(cbct, bad):
    kw = dict(synth.geom_kwargs(synth.CONFIGS["tiny"]))
    kw.update(bad)
    with pytest.raises(cbct.CbctError):
        cbct.Geometry(**kw)


def test_too_many_views_unsupported(cbct):
    kw = dict(synth.geom_kwargs(synth.CONFIGS["tiny"]), n_views=5000)
    with pytest.raises(cbct.CbctError, match="UNSUPPORTED"):
        cbct.Geometry(**kw)


@pytest.mark.parametrize("name", ["tiny", "small_halffan"])
def test_sample_count_matches_oracle(cbct, oracle_mod, name):
    """The library's analytic fp64 count equals the oracle's brute-force count."""
    kw = synth.geom_kwargs(synth.CONFIGS[name])
    assert cbct.Geometry(**kw).count_samples() == oracle_mod.count_samples(oracle_mod.Geom(**kw))


def test_sample_count_offcentre(cbct, oracle_mod):
    kw = dict(synth.geom_kwargs(synth.CONFIGS["tiny"]), vol_nx=20, vol_ny=27, vol_nz=13, vol_cx_mm=9.0,
              vol_cz_mm=-6.0, det_off_u_mm=30.0, det_off_v_mm=5.0, n_views=7, step_vox=0.3)
    assert cbct.Geometry(**kw).count_samples() == oracle_mod.count_samples(oracle_mod.Geom(**kw))


def test_slab_plan(cbct):
    kw = synth.geom_kwargs(synth.CONFIGS["large_512"])
    assert cbct.Geometry(**kw).num_slabs(4) == 1
    g = cbct.Geometry(**kw, max_workset_bytes=1 << 30)
    # per plane and 4 channels: (520 + 8) x 516 channel-interleaved cells (16 B for the 4 channels of a voxel; rows
    # padded to whole 128-B lines plus the skew) + 4 x 512 x 512 raw voxels (4 B);
    # two slab buffers, each with 2 * 2 border planes of packed cells, under 1 GiB
    packed, raw = 528 * 516 * 16, 4 * 512 * 512 * 4
    planes = ((1 << 30) // 2 - 4 * packed) // (packed + raw)
    assert g.num_slabs(4) == -(-512 // planes) == 9
    # 3 channels: one 16-B cell per voxel and channel (its four quarter-turn images; this geometry has that symmetry)
    packed3, raw3 = 3 * 528 * 516 * 16, 3 * 512 * 512 * 4
    assert g.num_slabs(3) == -(-512 // (((1 << 30) // 2 - 4 * packed3) // (packed3 + raw3)))
    assert g.num_slabs(1) > 1  # one channel in 16-B cells: 528 * 516^2 * 16 B = 2.2 GB does not fit
    assert cbct.Geometry(**kw, max_workset_bytes=3 << 30).num_slabs(1) == 1
    with pytest.raises(cbct.CbctError, match="NOMEM"):
        cbct.Geometry(**kw, max_workset_bytes=1 << 20).num_slabs(4)


def test_no_device_is_loud(cbct):
    """Without a CUDA device a compute call fails with CBCT_ERR_CUDA (no CPU fallback)."""
    try:
        import torch
        if torch.cuda.is_available():
            pytest.skip("a CUDA device is present")
    except ImportError:
        pass
    g = cbct.Geometry(**synth.geom_kwargs(synth.CONFIGS["tiny"]))
    with pytest.raises(cbct.CbctError, match="CUDA"):
        g.fp(np.zeros(g.n_vol, np.float32), np.zeros(g.n_sino, np.float32))


def test_missing_library_is_loud(cbct, monkeypatch, tmp_path):
    monkeypatch.setattr(cbct, "_lib", None)
    monkeypatch.setattr(cbct, "LIB_PATH", str(tmp_path / "nope.so"))
    with pytest.raises(cbct.CbctError, match="missing"):
        cbct.load_library()


@pytest.mark.parametrize("over", [dict(), dict(det_off_u_mm=115.0, det_nu=128, det_du_mm=1.6),
                                  dict(det_off_u_mm=-37.3, det_nu=77), dict(det_off_u_mm=400.0)])
def test_redundancy_weights_match_oracle(cbct, oracle_mod, over):
    """NEXT-1: the library's host table of w(u) (reading R12) equals the oracle's."""
    kw = dict(synth.geom_kwargs(synth.CONFIGS["tiny"]))
    kw.update(over)
    w = cbct.Geometry(**kw).redundancy_weights()
    assert np.max(np.abs(w - oracle_mod.redundancy_weight(oracle_mod.Geom(**kw)))) <= 1e-15
