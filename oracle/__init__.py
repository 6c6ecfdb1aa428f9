"""Float64 CPU oracle for the OSOG forward-render hot path.  TEST INFRASTRUCTURE ONLY:
importable from tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs;
never from paper_2606_21381_b200/.  See oracle/oracle.py and oracle/osog_oracle.c."""
