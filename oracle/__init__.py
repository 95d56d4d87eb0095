"""ORACLE package: plain, slow, FP64 CPU restatements of the paper's bound
definitions.  Test infrastructure only -- the product (paper_2607_01203_b200)
never imports it, and it never imports the product."""
