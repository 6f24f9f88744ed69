"""CPU oracle for the CAP routing-trace pipeline -- test infrastructure, not the product."""
