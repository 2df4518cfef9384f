"""Values the paper prints (tests/golden/paper_printed_values.txt, each with its PAPER.md line) against the host-side
definitions this repo uses: the throughput metric of bench.py (Eq. 17), the information throughput (Eq. 18), the
capacity / efficiency relation used to place the channel points (Eq. 3), the QC storage rule and Phi."""
import math
import os

import pytest

HERE = os.path.dirname(os.path.abspath(__file__))


def golden():
    vals = {}
    for line in open(os.path.join(HERE, "golden", "paper_printed_values.txt")):
        line = line.split("#", 1)[0].strip()
        if line:
            k, v = line.split("=")
            vals[k.strip()] = float(v)
    return vals


G = golden()


@pytest.mark.parametrize("code", ["q21", "q50", "random"])
def test_eq17_raw_throughput_matches_table2(code):
    import bench
    got = bench.decoded_mbit_per_s(G[f"t2_{code}_block_length_bits"], 1,
                                   G[f"t2_{code}_latency_ms"] * 1e-3 * G[f"t2_{code}_avg_iterations"])
    assert got == pytest.approx(G[f"t2_{code}_raw_mbit_s"], abs=1.5e-3)      # the table prints 3 decimals


@pytest.mark.parametrize("code", ["q21", "q50"])
def test_eq18_information_throughput_matches_table2(code):
    k_info = G[f"t2_{code}_raw_mbit_s"] * 1e3 * G[f"t2_{code}_code_rate"] * (1.0 - G[f"t2_{code}_fer"])
    assert k_info == pytest.approx(G[f"t2_{code}_info_kbit_s"], rel=3e-3)


def test_qc_code_stores_one_qth_of_the_edges():
    """P:499 / P:524: the lifted graph of a QC code has q x (stored connections) edges; for the paper's ensemble that
    is the random code's edge count up to the rounding of the base graph."""
    for code in ("q50", "q21"):
        lifted = G[f"t2_{code}_connections"] * G[f"t2_{code}_expansion"]
        assert lifted == pytest.approx(G["t2_random_connections"] * (1.008 if code == "q21" else 1.0), rel=1e-3)


def test_beta_at_table4_operating_point():
    from oracle import capacity
    beta = G["t4_rate"] / (0.5 * math.log2(1.0 + G["t4_snr"]))
    assert beta == pytest.approx(G["t4_beta"], abs=5e-3)
    # the oracle's Shannon helper inverts the same relation: sigma* at rate C(s) is 1/sqrt(s)
    c = 0.5 * math.log2(1.0 + G["t4_snr"])
    assert capacity.shannon_sigma_star(c) == pytest.approx(1.0 / math.sqrt(G["t4_snr"]), rel=1e-12)
    # and the BIAWGN capacity at that SNR is below the unconstrained one, by little at such low SNR
    c_bi = capacity.biawgn_capacity(1.0 / math.sqrt(G["t4_snr"]))
    assert 0.97 * c < c_bi < c


def test_phi_is_its_own_inverse(oracle_lib):
    for x in (0.01, 0.3, 1.0, 4.0, 12.0):
        assert oracle_lib.phi(oracle_lib.phi(x)) == pytest.approx(x, rel=1e-10)
        assert oracle_lib.phi(x) == pytest.approx(-math.log(math.tanh(x / 2.0)), rel=1e-9)
