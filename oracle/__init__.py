"""fp64 CPU oracle of the arXiv 1507.04941 hot path -- TEST INFRASTRUCTURE ONLY (see pgsf_oracle.c)."""
