"""CPU oracle -- TEST INFRASTRUCTURE ONLY (see orc.h).  Never imported by the product."""
