"""The seeded edge-case generators used by the GPU parity tests produce descriptors that the
library accepts (no device needed for the validation) and that the oracle can advance."""
import numpy as np
import pytest

from paper_1408_5853_b200 import inputs as I


@pytest.mark.parametrize("nr,nz,batch,poly", [(128, 14, 2, True), (512, 24, 3, False), (512, 9, 5, True),
                                              (1024, 21, 2, False), (2048, 13, 2, True), (8192, 6, 1, False)])
def test_band_spec_is_a_valid_descriptor(nr, nz, batch, poly):
    from paper_1408_5853_b200 import binding
    from oracle.heat_oracle import Oracle
    s = I.band_spec(nr + nz, nr=nr, nz=nz, batch=batch, poly_laws=poly)
    seg = s["seg_layer"]
    assert seg.shape == (batch, nr - 1) and seg.dtype == np.uint8
    for b in range(batch):
        nodes = np.flatnonzero(np.diff(seg[b].astype(int))) + 1       # interface nodes
        assert len(nodes) == len(s["layers"]) - 1
        assert nodes[0] >= 2 and nodes[-1] <= nr - 3 and np.all(np.diff(nodes) >= 2)
        assert np.all(np.bincount(nodes // 8) <= 1)                   # one interface node per 8-node chunk
    assert binding.heat_workspace_bytes(s) > 0                        # the library's own validation
    lim = binding.heat_stable_dt(s)
    assert lim > 0
    s = dict(s, dt=0.8 * lim)
    o = Oracle(s)
    o.step(3)
    assert np.all(np.isfinite(o.field(batch - 1)))


def test_band_spec_is_seeded():
    a, b, c = I.band_spec(5, nr=512, nz=12), I.band_spec(5, nr=512, nz=12), I.band_spec(6, nr=512, nz=12)
    assert np.array_equal(a["T_init"], b["T_init"]) and np.array_equal(a["seg_layer"], b["seg_layer"])
    assert not np.array_equal(a["T_init"], c["T_init"])
