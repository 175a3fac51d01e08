"""fp64 CPU oracle of the cp4d hot path.  TEST INFRASTRUCTURE ONLY (see cp4d_ref.c header)."""
