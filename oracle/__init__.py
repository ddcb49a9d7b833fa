"""ORACLE -- TEST INFRASTRUCTURE, NOT PRODUCT CODE.  See cn_oracle.py / cn_thomas.c / nshape_table1.py."""
