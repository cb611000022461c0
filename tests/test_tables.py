"""The product's numpy table builder against the oracle's long-double builder."""
import numpy as np
import pytest

from paper_2209_15445_b200.inputs import materials


@pytest.mark.parametrize("name", ["Pb", "LAr", "Si", "PbWO4", "vacuum"])
def test_product_tables_match_oracle(ob, name):
    m = materials.standard_materials()[name]
    tab = materials.build_tables(m)
    scal = materials.material_scalars(m)
    otab, oscal = ob.build_material(m.Z, m.A, m.rho)
    np.testing.assert_allclose(scal[:6], oscal[:6], rtol=1e-11)
    # Klein-Nishina loses ~1e-10 to cancellation in plain fp64 near kappa = 2e-3 (SURVEY.md M7 note)
    np.testing.assert_allclose(tab[0], otab[0], rtol=5e-10)
    np.testing.assert_allclose(tab[1:], otab[1:], rtol=1e-11, atol=1e-300)


def test_survey_cut_values():
    """M4 values computed while surveying: Pb 1.0225/0.1744, LAr 0.2625/0.0175, Si 0.4063/0.0157 MeV."""
    std = materials.standard_materials()
    want = {"Pb": (1.0225, 0.1744), "LAr": (0.2625, 0.0175), "Si": (0.4063, 0.0157), "PbWO4": (0.8115, 0.1411)}
    for name, (te, kg) in want.items():
        e, g = materials.compute_cuts(std[name])
        assert e == pytest.approx(te, abs=6e-5) and g == pytest.approx(kg, abs=6e-5)
