"""Test-infrastructure oracles (fp64 CPU).  Never imported by the product path."""
