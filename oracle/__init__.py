"""ORACLE — TEST INFRASTRUCTURE ONLY.

Plain CPU implementation of the Shan-Chen LBM step written from the paper
(oracle/lbm_oracle.cpp) plus the Maxwell construction (oracle/maxwell.py).
Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline /
--impl reference legs may import this package.
"""
