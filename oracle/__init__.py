"""ORACLE -- test infrastructure only.  See shaken_oracle.c for the paper citations.
Nothing under paper_1908_07341_b200/ may import this package."""
