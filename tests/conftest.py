import os
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)


def pytest_configure(config):
    config.addinivalue_line("markers", "gpu: needs a CUDA device (run on the B200 box with -m gpu)")


@pytest.fixture(scope="session")
def cfg0():
    """Config 0 of BASELINE.json (tiny phantom), generated once on the CPU, as numpy arrays."""
    import synth
    ph = synth.generate(synth.config_spec(0), device="cpu")
    return ph


def as_np(ph):
    """Numpy views of a Phantom's arrays (COO copied to host if needed)."""
    return dict(
        vox=ph.coo_voxel.cpu().numpy(), beam=ph.coo_beamlet.cpu().numpy(), val=ph.coo_val.cpu().numpy(),
        n_v=ph.n_voxels, n_b=ph.n_beamlets, sid=ph.voxel_struct.numpy(), T=ph.struct_T.numpy(),
        wo=ph.struct_w_over.numpy(), wu=ph.struct_w_under.numpy(),
        lco=ph.leafrow_col_offset.numpy(), aro=ph.angle_row_offset.numpy(), aco=ph.angle_col_offset.numpy(),
    )
