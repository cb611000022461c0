import os
import sys

import numpy as np
import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)


def pytest_configure(config):
    config.addinivalue_line("markers", "gpu: needs a CUDA device (run on the B200 box)")


@pytest.fixture(scope="session")
def calo():
    from paper_2209_15445_b200.inputs import geometry, materials
    g = geometry.calorimeter()
    mats, tabs, scal = materials.build_material_set(g.material_names)
    return g, mats, tabs, scal


@pytest.fixture(scope="session")
def barrel_patch():
    """A 12 x 12 crystal patch of the barrel (same crystals, Si shells and mother volume)."""
    from paper_2209_15445_b200.inputs import geometry, materials
    g = geometry.barrel(n_eta=12, n_phi=12)
    mats, tabs, scal = materials.build_material_set(g.material_names)
    return g, mats, tabs, scal


@pytest.fixture(scope="session")
def barrel_patch_compound():
    """The same patch with crystals of the real compound PbWO4 (Pb + W + 4 O) and its element-selector tables."""
    from paper_2209_15445_b200.inputs import geometry, materials
    g = geometry.barrel(n_eta=12, n_phi=12, crystal="PbWO4_true")
    mats, tabs, scal = materials.build_material_set(g.material_names)
    return g, mats, tabs, scal, materials.element_tables(mats)


@pytest.fixture(scope="session")
def barrel_full():
    from paper_2209_15445_b200.inputs import geometry, materials
    g = geometry.barrel()
    mats, tabs, scal = materials.build_material_set(g.material_names)
    return g, mats, tabs, scal


@pytest.fixture(scope="session")
def ob():
    from oracle import binding
    return binding
