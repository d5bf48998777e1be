"""CPU oracle of the cone-beam FBS hot path -- test infrastructure, not product code."""
