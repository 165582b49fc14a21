"""fp64 CPU oracle — TEST INFRASTRUCTURE ONLY (see allegro_oracle.py header).  Never imported by the
product package `paper_2304_10061_b200`."""
