"""CPU oracle (test infrastructure only; see the headers of the modules in this package)."""
