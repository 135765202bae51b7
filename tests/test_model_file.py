"""Front end for the paper's model-file format (Table 4): the paper's own example must
parse to exactly the Lotka-Volterra network of BASELINE config 2."""
import math
import os

import numpy as np
import pytest

import rt_workloads as W
from paper_2103_00405_b200.model_file import ModelFileError, load_model, parse_model

HERE = os.path.dirname(os.path.abspath(__file__))


def test_paper_table4_example_is_config2():
    m = load_model(os.path.join(HERE, "golden", "lotka_table4.model"))
    ref, x0 = W.lotka_volterra()
    assert m["species"] == ["A", "B"] and m["t_end"] == 2.0 and m["max_firings"] == 10000
    np.testing.assert_array_equal(m["x0"], x0)
    for key in ("react_ptr", "react_species", "react_sigma", "stoich_ptr", "stoich_species", "stoich_v", "rate"):
        np.testing.assert_array_equal(m["net"][key], ref[key], err_msg=key)
        assert m["net"][key].dtype == ref[key].dtype
    assert m["net"]["n_species"] == 2 and m["net"]["n_reactions"] == 3


def test_dimerisation_and_catalyst_forms():
    m = parse_model("# init\nA = 5\nC = 1\nD = 0\n# reactions\n1 A 1 A - -> 1 D : 0.5\n2 A 1 C - -> 1 C 1 D : 2\n# end\n")
    net = m["net"]
    assert list(net["react_sigma"]) == [2, 2, 1]                 # "1 A 1 A" == "2 A": sigma = 2
    assert list(net["stoich_species"][:2]) == [0, 2] and list(net["stoich_v"][:2]) == [-2, 1]
    assert list(net["stoich_species"][2:]) == [0, 2]             # the catalyst C has no net change
    assert m["t_end"] == math.inf and m["max_firings"] == 0


@pytest.mark.parametrize("text", [
    "# init\nA = 1\n# reactions\n1 Z - -> NULL : 1\n",          # unknown species
    "# init\nA = 1\n# reactions\n1 A -> NULL : 1\n",            # wrong arrow
    "# init\nA = 1\n# reactions\n0 A - -> NULL : 1\n",          # coefficient < 1
    "# init\nA = 1\n# reactions\n1 A - -> NULL : fast\n",       # rate not a number
    "# init\nA = x\n# reactions\n1 A - -> NULL : 1\n",          # count not an integer
    "# init\nA = 1\nA = 2\n# reactions\n1 A - -> NULL : 1\n",  # species twice
    "# init\nA = 1\n",                                             # no reactions
    "A = 1\n",                                                      # text before a section
])
def test_malformed_files_are_rejected(text):
    with pytest.raises(ModelFileError):
        parse_model(text)


@pytest.mark.gpu
def test_parsed_model_runs_and_matches_oracle():
    import oracle
    import paper_2103_00405_b200 as rt
    m = load_model(os.path.join(HERE, "golden", "lotka_table4.model"))
    o = oracle.run(m["net"], m["x0"], 3, 0, m["max_firings"], m["t_end"], m["max_firings"])
    with rt.Model(m["net"]) as model:
        g = model.run(m["x0"], 3, 0, m["max_firings"], m["t_end"], m["max_firings"])
    np.testing.assert_array_equal(g["trace_mu"], o["trace_mu"])
    np.testing.assert_array_equal(g["x"], o["x"])
    assert g["stop"] == o["stop"] and g["firings"] == o["firings"]
