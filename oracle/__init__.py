"""CPU oracle for UniFrac -- TEST INFRASTRUCTURE ONLY (see oracle/unifrac_oracle.c header).

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may
import this package.  It imports nothing from paper_2107_05397_b200."""
