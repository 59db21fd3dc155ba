"""fp64 CPU oracle -- TEST INFRASTRUCTURE, not product code (see oracle/qxd_ref.cpp header)."""
