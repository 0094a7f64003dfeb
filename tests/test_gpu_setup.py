"""S0 on the device (vpmc_setup.cuh): the packed opening bitmap and the two safe-distance maps built by kernels from the
caller's uint8 bitmap, against plain definitions: numpy's packbits and scipy's chessboard distance transform (a library
routine, so the check shares nothing with the kernels).  Also the RED-ceiling measurement kernel."""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu


def _engine_with_bitmap(op, pitch=0.1):
    from paper_2307_01416_b200 import binding, workloads as wl
    w = wl.small_water(n=(8, 8, 20), with_aperture=True)
    ny, nx = op.shape
    w["beams"][0]["aperture"] = wl.aperture(op, -0.5 * nx * pitch, -0.5 * ny * pitch, pitch, pitch, 30.0, 40.0)
    return binding.Engine(w)


def _reference_tables(op):
    from scipy.ndimage import distance_transform_cdt
    ny, nx = op.shape
    rw = (nx + 31) // 32
    padded = np.zeros((ny, rw * 32), dtype=np.uint8)
    padded[:, :nx] = op != 0
    bits = np.packbits(padded, axis=1, bitorder="little").view(np.uint32).reshape(ny, rw)
    # distance to the nearest pixel that is not open, everything outside the bitmap being brass: pad by one ring of zeros
    p = np.zeros((ny + 2, nx + 2), dtype=np.uint8)
    p[1:-1, 1:-1] = op != 0
    d_br = distance_transform_cdt(p, metric="chessboard")[1:-1, 1:-1]
    # distance to the nearest open pixel (none outside)
    if (op != 0).any():
        d_op = distance_transform_cdt((op == 0).astype(np.uint8), metric="chessboard")
    else:
        d_op = np.full(op.shape, 255)
    return bits, np.minimum(d_br, 255).astype(np.uint8), np.minimum(d_op, 255).astype(np.uint8)


@pytest.mark.parametrize("shape", ["disc", "star", "ragged", "closed", "open", "far"])
def test_device_built_aperture_tables_match_their_definitions(shape):
    from paper_2307_01416_b200 import workloads as wl
    rng = np.random.default_rng(11)
    if shape == "disc":
        op = wl.disc_bitmap(128, 0.1, 3.0)[0]
    elif shape == "star":
        op = wl.config5()["beams"][0]["aperture"]["open"]          # 1024^2, the bench's irregular opening
    elif shape == "ragged":                                          # sizes that are no multiple of 32, random blobs, open pixels on the rim
        op = (rng.random((77, 109)) < 0.7).astype(np.uint8)
        op[20:50, 30:90] = 1
        op[0, :] = 1
    elif shape == "closed":
        op = np.zeros((64, 96), dtype=np.uint8)
    elif shape == "open":
        op = np.ones((40, 33), dtype=np.uint8)
    else:                                                            # distances beyond the 255 cap
        op = np.zeros((700, 640), dtype=np.uint8)
        op[:, :320] = 1
        op[5, 600] = 1
    eng = _engine_with_bitmap(op)
    bits, dist = eng.aperture_tables(0)
    rb, d_br, d_op = _reference_tables(op)
    assert np.array_equal(bits, rb)
    assert np.array_equal(dist[0], d_br)
    assert np.array_equal(dist[1], d_op)
    eng.close()


def test_tables_follow_a_replaced_bitmap():
    """set_aperture on a live handle releases the old tables and builds new ones; a dose before and after runs."""
    from paper_2307_01416_b200 import binding, workloads as wl
    import ctypes as C
    w = wl.small_water(n=(8, 8, 20), with_aperture=True)
    eng = binding.Engine(w)
    d0 = eng.dose(2000, 3).cpu().numpy()
    op = np.zeros((64, 64), dtype=np.uint8)
    eng._check(binding.lib().vpmc_set_aperture(eng._h, 0, 30.0, binding.BRASS, op.ctypes.data, 64, 64, C.c_float(-3.2), C.c_float(-3.2),
                                               C.c_float(0.1), C.c_float(0.1), C.c_float(40.0)))
    d1 = eng.dose(2000, 3).cpu().numpy()
    assert d0.sum() > 0 and d1.sum() == 0.0                            # closed block: nothing reaches the CT (70 MeV, P7)
    _, dist = eng.aperture_tables(0)
    assert (dist[1] == 255).all() and (dist[0] == 0).all()
    eng.close()


def test_red_ceiling_measurement_runs_and_counts():
    from paper_2307_01416_b200 import binding, workloads as wl
    eng = binding.Engine(wl.small_water(n=(8, 8, 20)))
    rate, n = eng.bench_red(4 << 20, 1 << 28)
    assert n >= (1 << 27) and 1e9 < rate < 1e13
    eng.close()
