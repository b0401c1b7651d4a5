"""CPU oracle -- test infrastructure only (see the module headers).  Never imported by the product path."""
