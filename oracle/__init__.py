"""fp64 CPU oracle of the ELDR decode-MoE hot path -- test infrastructure, not the product."""
