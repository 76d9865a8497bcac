"""The seeded input generators that serve both the oracle and the CUDA path (synth/): the torch recipe used for
the large on-device workloads must reproduce the numpy recipe bit for bit."""
import numpy as np

import synth


def test_hash_visibilities_torch_is_bit_identical():
    a = synth.hash_visibilities(np.arange(301), 13, 1003)
    b = synth.hash_visibilities_torch(301, 13, 1003, "cpu", chunk_rows=64).numpy()
    assert np.array_equal(a.view(np.uint32), b.view(np.uint32))
    # a subset regenerated on its own (what the full-size parity tests feed the oracle)
    rows = np.array([5, 17, 300])
    sub = synth.hash_visibilities(rows, 4, 1003, n_chan_total=13, chan0=6)
    assert np.array_equal(sub.view(np.uint32), np.ascontiguousarray(b[rows][:, 6:10]).view(np.uint32))
