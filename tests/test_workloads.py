"""Input generators (paper_2001_05234_b200/workloads.py): grid of eq. 7 and the seeded fields."""
import math

import numpy as np
import torch

from paper_2001_05234_b200 import workloads as wl


def test_tanh_grid_closed_form_properties():
    for nz, lz, a in [(32, 2.0, 1.6), (128, 2.0, 1.5), (512, 2.0, 2.0)]:
        dzc, dzf, zc = wl.tanh_grid(nz, lz, a)
        assert dzc.shape == (nz + 1,) and dzf.shape == (nz,)
        assert abs(float(dzf.sum()) - lz) < 1e-14
        assert torch.all(dzf > 0) and torch.all(dzc > 0)
        # symmetric about the mid-plane, clustered at the walls
        assert torch.max(torch.abs(dzf - dzf.flip(0))) < 1e-14
        assert dzf[0] < dzf[nz // 2]
        # eq. 7 evaluated at the face coordinates Z = m/nz
        m = nz // 4
        zf_m = 0.5 * (1 + math.tanh(a * (m / nz - 0.5)) / math.tanh(a / 2)) * lz
        assert abs(float(dzf[:m].sum()) - zf_m) < 1e-14
        assert float(dzc[0]) == float(dzf[0]) and float(dzc[nz]) == float(dzf[nz - 1])
        assert abs(float(dzc[1:nz].sum()) - float(zc[-1] - zc[0])) < 1e-14


def test_fields_are_seeded_and_shaped():
    a = wl.make_workload("C2", n_override=(32, 16, 24))
    b = wl.make_workload("C2", n_override=(32, 16, 24))
    f = a.fields["f"]
    assert f.shape == (24, 16, 32) and f.dtype == torch.float64
    assert torch.equal(f, b.fields["f"])
    # volume-weighted mean removed (reading S3)
    assert abs(float((f * a.dzf[:, None, None]).sum())) < 1e-10
    c1 = wl.make_workload("C1")
    assert abs(float(c1.fields["f"].mean())) < 1e-15 and float(c1.fields["f"].abs().max()) <= 1.05


def test_c5_recipe_small():
    w = wl.make_workload("C5", n_override=(64, 48, 32))
    u, v, ww = w.fields["u"], w.fields["v"], w.fields["w"]
    assert w.dt == 1e-4 and w.kind == "projection"
    assert torch.all(ww[-1] == 0)
    # bulk velocity of the Poiseuille part is ~1 (fluctuations have zero mean)
    ub = float((u.mean(dim=(1, 2)) * w.dzf).sum() / w.dzf.sum())
    assert abs(ub - 1.0) < 0.05
    # spectrum decays: energy in the lowest wavenumber shell exceeds the highest
    vh = torch.fft.rfftn(v).abs() ** 2
    assert float(vh[1, 1, 1]) > float(vh[12, 20, 28])
    assert np.isfinite(float(u.sum()))
