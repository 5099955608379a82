"""bench.py's second CPU figure (`cpu_fft_baseline`) is a restatement of the C5 step with scipy.fft; before its time is
quoted next to the oracle's it has to compute the same thing.  Checked here against the oracle on a small periodic-x/y,
Neumann-z, stretched grid."""
import numpy as np

import bench
from oracle import cans_oracle as orc
from paper_2001_05234_b200 import workloads as wl


def test_cpu_fft_projection_matches_the_oracle():
    nx, ny, nz = 32, 24, 11
    lx, ly, lz = 2 * np.pi, np.pi, 2.0
    dzc_t, dzf_t, _ = wl.tanh_grid(nz, lz, 1.6)
    dzc, dzf = dzc_t.numpy(), dzf_t.numpy()
    rng = np.random.default_rng(3)
    u, v, w = (rng.standard_normal((nz, ny, nx)) for _ in range(3))
    w[-1] = 0.0                                         # the top wall face carries no flow (compatibility of the Neumann problem)
    dt = 1e-2
    bc = (("P", "P"), ("P", "P"), ("N", "N"))
    un, vn, wn, phi, _ = orc.projection(u, v, w, dt, lx, ly, lz, bc, dzc, dzf)
    got = bench.cpu_fft_projection(u, v, w, dt, lx, ly, lz, dzc, dzf, workers=2)
    for g, r, name in zip(got, (un, vn, wn, phi), ("u", "v", "w", "Phi")):
        assert np.linalg.norm(g - r) <= 1e-11 * np.linalg.norm(r), name


def test_both_cpu_legs_time_the_same_slab():
    import inspect
    assert bench.NZ_SAMPLE >= 32
    assert "NZ_SAMPLE" in inspect.getsource(bench.run_reference)
    assert inspect.getsource(bench.run_ours).count("nz_sample = NZ_SAMPLE") == 1
