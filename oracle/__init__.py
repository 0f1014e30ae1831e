"""CPU oracle (test infrastructure).  See oracle/gst_oracle.hpp for what it is and who may call it."""
