"""The seeded input generator (cubegen/): Philox integers against the published known-answer
vectors, CPU and CUDA-source restatements against each other, and the structure of the configs."""
import numpy as np

import cubegen


def test_philox_known_answers():
    # Random123 kat_vectors for philox4x32-10
    w = cubegen.philox4x32_10(0, 0, 0, 0, 0, 0)
    assert [int(x) for x in w] == [0x6627E8D5, 0xE169C58D, 0xBC57AC4C, 0x9B00DBD8]
    f = 0xFFFFFFFF
    w = cubegen.philox4x32_10(f, f, f, f, f, f)
    assert [int(x) for x in w] == [0x408F276D, 0x41C83B0E, 0xA20BC7C6, 0x6D5451FD]
    w = cubegen.philox4x32_10(0x243F6A88, 0x85A308D3, 0x13198A2E, 0x03707344, 0xA4093822, 0x299F31D0)
    assert [int(x) for x in w] == [0xD16CFE09, 0x94FDCCEB, 0x5001E420, 0x24126EA1]


def test_philox_cuda_source_matches_numpy():
    rng = np.random.default_rng(0)
    for _ in range(20):
        c = [int(v) for v in rng.integers(0, 2 ** 32, 6)]
        assert cubegen.philox_device_words(*c) == tuple(int(x) for x in cubegen.philox4x32_10(*c))


def test_config_structure_small():
    c1 = cubegen.scaled("c1", (48, 40, 32), nsrc=4)
    a = cubegen.generate_numpy(c1)
    assert a.shape == (32, 40, 48) and a.dtype == np.float32 and not np.isnan(a).any()
    assert (a == cubegen.generate_numpy(c1)).all()                           # deterministic
    a0 = cubegen.generate_numpy(cubegen.scaled("c1", (48, 40, 32), nsrc=0))
    assert abs(float(a0.std()) - 1.0) < 0.02 and abs(float(a0.mean())) < 0.02  # N(0,1) noise
    assert a.max() > 30.0 and (a >= a0 - 1e-6).all()                         # + positive sources
    c2 = cubegen.scaled("c2", (16, 16, 1024), nsrc=2)
    planes = cubegen.nan_planes(c2)
    b = cubegen.generate_numpy(c2)
    assert 2 <= len(planes) <= 30
    assert int(np.isnan(b).sum()) == len(planes) * 16 * 16 and np.isnan(b[planes]).all()
    c3 = cubegen.scaled("c3", (32, 32, 64))
    assert 0.002 < float(np.isnan(cubegen.generate_numpy(c3)).mean()) < 0.01
    c4 = cubegen.scaled("c4", (64, 64, 8))
    d = cubegen.generate_numpy(c4)
    assert 0.27 < float((d == 0).mean()) < 0.33 and len(np.unique(d)) <= 4097 and d.min() == 0.0


def test_bricks_tile_the_cube():
    c = cubegen.scaled("c5", (32, 32, 32), nsrc=6)
    full = cubegen.generate_numpy(c)
    for oz in (0, 16):
        for oy in (0, 16):
            for ox in (0, 16):
                br = cubegen.generate_numpy(c, origin=(ox, oy, oz), brick=(16, 16, 16))
                ref = full[oz:oz + 16, oy:oy + 16, ox:ox + 16]
                assert np.allclose(br, ref, rtol=0, atol=1e-6)
