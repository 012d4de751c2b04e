"""CPU oracle (test infrastructure only; see oracle/lra_ref.c).  Never imported by the product."""
