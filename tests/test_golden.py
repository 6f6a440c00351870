"""tests/golden: the numbers the paper states against the build's defaults, and the stored oracle outputs against the
oracle as it stands (see tests/golden/README.md)."""
import importlib.util
import inspect
import os

from oracle import peel as OP
from paper_1908_01949_b200 import binding as B, synth

GOLDEN = os.path.join(os.path.dirname(os.path.abspath(__file__)), "golden")


def _constants():
    out = {}
    for line in open(os.path.join(GOLDEN, "paper_constants.txt")):
        if line.startswith("#") or not line.strip():
            continue
        name, value, unit, cite, use = [x.strip() for x in line.split("|")]
        assert int(cite) > 0
        out[name] = float(value)
    return out


def test_defaults_equal_the_numbers_the_paper_states():
    c = _constants()
    assert synth.P_SIGNAL == c["signal_momentum"]
    assert synth.make_uniform_field().bz_T == c["field"]
    g = synth.make_geometry()
    assert len(g.r_mm) == c["sense_layers"] and g.R0_mm == c["seed_radius_R0"]
    sig = inspect.signature(B.cdc_refine_tracks).parameters
    assert sig["n_iterations"].default == c["refinement_iterations"]
    assert inspect.signature(B.cdc_peel_turns).parameters["min_hits"].default == c["stop_unclassified_hits"]   # :83
    assert inspect.signature(OP.peel).parameters["min_hits"].default == c["stop_unclassified_hits"]
    import test_peel                                                                # the half-widths the peeling tests use
    assert test_peel.HALF_WIDTH == [c["hough_resolution_theta"], c["extrapolation_resolution_z0"],
                                    c["hough_resolution_pxy"], c["hough_resolution_pxy"], c["extrapolation_resolution_pz0"]]


def test_oracle_reproduces_its_stored_outputs_bit_for_bit():
    spec = importlib.util.spec_from_file_location("make_golden", os.path.join(GOLDEN, "make_golden.py"))
    mod = importlib.util.module_from_spec(spec)
    spec.loader.exec_module(mod)
    assert mod.compute() == open(os.path.join(GOLDEN, "oracle_cfg0_scan.txt")).read()
