"""CPU oracle (test infrastructure only): see oracle/tfo.c."""
