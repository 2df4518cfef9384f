"""ORACLE (test infrastructure): prints the sigma* table stored in paper_1702_07740_b200/workloads.py:SIGMA_STAR.

Run `python -m oracle.make_sigma_table` from the repo root; it calls only oracle/capacity.py.  The digits it prints
are pasted into workloads.py (the generator module must not import oracle/); tests/test_capacity.py checks that the
stored table equals a fresh computation.
"""
from oracle.capacity import sigma_star, sigma_for_gap

if __name__ == "__main__":
    for rate in (0.1, 0.05, 0.02):
        print(f"    {rate}: {sigma_star(rate):.10f},")
    for rate, gap in ((0.1, 1.5), (0.1, 0.5), (0.02, 0.3)):
        print(f"# rate {rate} +{gap} dB: sigma = {sigma_for_gap(rate, gap):.8f}")
    for gap in (0.1, 0.3, 0.5, 0.7, 0.9, 1.1):
        print(f"# rate 0.05 +{gap} dB: sigma = {sigma_for_gap(0.05, gap):.8f}")
