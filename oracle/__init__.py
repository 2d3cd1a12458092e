"""CPU oracle of the unpack + three-threshold clustering path.  TEST INFRASTRUCTURE ONLY:
see the header of sst_oracle.c.  Nothing under paper_2101_11489_b200/ imports this package."""
