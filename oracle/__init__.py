"""ORACLE — test infrastructure (fp64 CPU, from the paper). Not product code; see oracle.py."""
