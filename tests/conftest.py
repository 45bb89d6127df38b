import os
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)


def pytest_configure(config):
    config.addinivalue_line("markers", "gpu: needs a CUDA device (run on the B200 box)")


@pytest.fixture(scope="session")
def cfg0_oracle():
    """Oracle loaded with BASELINE config 0 (mesh, equilibrium, species, both fields)."""
    from oracle import Oracle
    from paper_2606_24327_b200 import synth

    cfg = synth.CONFIGS[0]
    RZ, tri = synth.make_mesh(cfg)
    o = Oracle()
    o.equilibrium_set(**synth.equilibrium_args(cfg))
    o.species_set(**synth.species_args(cfg))
    o.mesh_load(RZ, tri, cfg.n_planes, cfg.phi_period)
    dphi, dap = synth.make_fields(cfg, RZ)
    o.fields_set(0, dphi)
    o.fields_set(1, dap)
    return cfg, RZ, tri, o, (dphi, dap)
