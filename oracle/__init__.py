"""ORACLE — test infrastructure only (CPU fp64 restatement of the hot path, written from the paper).

Nothing in the product package imports this; see oracle/README.md.
"""
