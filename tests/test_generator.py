"""Seeded input generator (tpcsynth): determinism and the edge cases the parity tests rely on.  No tracker arithmetic."""
import numpy as np

import tpcsynth


def test_same_seed_same_bytes_and_other_seed_differs():
    a = tpcsynth.generate(1, n_tracks=300)
    b = tpcsynth.generate(1, n_tracks=300)
    c = tpcsynth.generate(1, n_tracks=300, seed=a.seed + 1)
    for s in range(36):
        for f in ("y", "z", "row", "label"):
            assert np.array_equal(getattr(a, f)[s], getattr(b, f)[s])
    assert a.n_clusters != c.n_clusters or not np.array_equal(a.y[0], c.y[0])


def test_time_frame_without_collisions_is_empty():
    tf = tpcsynth.generate(2, n_orbits=1, coll_times=[])
    assert tf.n_sectors == 36 and tf.n_clusters == 0 and all(a.shape == (0,) for a in tf.row)


def test_hand_placed_collisions_keep_the_full_axis():
    T = 128 * tpcsynth.ORBIT_US
    tf = tpcsynth.generate(3, coll_times=[0.0, T], coll_mult=200)
    assert tf.coll_t.tolist() == [0.0, T] and tf.trk_coll.shape[0] == 400
    zmax = max(float(z.max()) for z in tf.z if z.size)
    assert 29_000.0 < zmax <= tf.params.z_hi and tf.params.z_hi > 29_600.0
    rows = np.concatenate(tf.row)
    assert rows.max() <= 151 and tf.params.n_rows == 152
