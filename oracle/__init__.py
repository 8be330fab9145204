"""ORACLE — test infrastructure, not product code.  See oracle/lgo.h."""
