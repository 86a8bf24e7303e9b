"""Seeded input generator (paper_1105_4747_b200/inputs.py): determinism, slab independence,
statistics of the recipe in DESIGN.md "Input recipe".  CPU only."""
import numpy as np
import torch

from paper_1105_4747_b200 import inputs
from paper_1105_4747_b200.workloads import WORKLOADS, scaled


def test_philox_known_answer():
    # Philox4x32-10 known-answer vectors of Salmon et al. 2011 (Random123 kat_vectors)
    z = torch.zeros(1, dtype=torch.int64)
    out = inputs.philox4x32(z, z, z, z, 0, 0)
    assert [int(x) for x in out] == [0x6627E8D5, 0xE169C58D, 0xBC57AC4C, 0x9B00DBD8]
    f = torch.full((1,), 0xFFFFFFFF, dtype=torch.int64)
    out = inputs.philox4x32(f, f, f, f, 0xFFFFFFFF, 0xFFFFFFFF)
    assert [int(x) for x in out] == [0x408F276D, 0x41C83B0E, 0xA20BC7C6, 0x6D5451FD]


def test_fields_deterministic_and_slab_independent():
    w = scaled(WORKLOADS[1], 32)
    a = inputs.make_fields(w)
    b = inputs.make_fields(w)
    assert torch.equal(a["delta"], b["delta"]) and torch.equal(a["v_pec"][0], b["v_pec"][0])
    s = inputs.make_fields(w, z0=5, z1=9)
    assert torch.allclose(s["delta"], a["delta"][5:9], rtol=0, atol=1e-6)
    assert torch.allclose(s["v_pec"][0], a["v_pec"][0][5:9], rtol=0, atol=1e-4)
    assert a["delta"].dtype == torch.float32 and a["delta"].shape == (32, 32, 32)


def test_field_statistics():
    w = WORKLOADS[1]
    f = inputs.make_fields(w)
    d = f["delta"].double().numpy()
    v = f["v_pec"][0].double().numpy()
    assert d.min() > -1.0
    g = np.log1p(d) + 0.5 * w.sigma_g ** 2
    assert abs(g.std() / w.sigma_g - 1) < 0.05 and abs(g.mean()) < 0.05
    assert abs(v.std() / w.sigma_v - 1) < 0.05 and abs(v.mean()) < 0.05 * w.sigma_v
    # different fields are independent draws
    assert abs(np.corrcoef(g.ravel(), v.ravel())[0, 1]) < 0.05
