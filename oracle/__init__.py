"""Oracle package: TEST INFRASTRUCTURE ONLY (see oracle/olsm.c header). Never imported by the product path."""
