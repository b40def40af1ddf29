"""CPU oracle (test infrastructure only).  See ia_oracle.cpp.  Nothing under
``paper_2509_15117_b200`` may import this package, and this package imports nothing from it."""
