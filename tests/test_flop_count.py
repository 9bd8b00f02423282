"""The algorithmic flop counts behind bench.py's roofline, pinned by running the oracle's
own formulas on a counting scalar type (oracle/flop_count.cpp).  CPU only."""
import os

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def golden():
    out = {}
    for line in open(os.path.join(ROOT, "tests", "golden", "flop_counts.txt")):
        if line.startswith("#") or not line.strip():
            continue
        k, v = line.split()
        out[k] = int(v)
    return out


def test_counts_match_the_stored_ones():
    from oracle import flop_count
    assert flop_count.counts() == golden()


def test_bench_uses_a_count_that_does_not_exceed_the_oracle_formulation():
    """bench.py's numerators are SURVEY 8(d)'s textbook counts with shared subexpressions; they must not exceed
    what the oracle's formulas, written out literally, actually execute (else the roofline fraction would be
    inflated), and they must be of the same size (within a factor 1.6)."""
    import bench
    g = golden()
    for scheme, key in (("weno5", "weno5"), ("weno7", "weno7"), ("musta", "musta")):
        per_L, per_step = bench.FLOPS_PER_CELL_L[scheme], bench.FLOPS_PER_CELL_STEP[scheme]
        assert per_L <= g["L_" + key] <= 1.6 * per_L, (scheme, per_L, g["L_" + key])
        assert per_step <= g["step_" + key] <= 1.6 * per_step
        assert abs(per_step - (3 * per_L + 60)) <= 1
    # the pieces: one WENO reconstruction has 3 (4) sub-stencils with one division each for alpha and omega
    assert g["weno5"] > 60 and g["weno7"] > g["weno5"]
    assert g["L_weno5"] == g["con2prim"] + 3 * g["signal_speed"] + 3 * (g["phys_flux"] + g["llf_split_weno5"] + 10)
