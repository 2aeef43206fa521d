"""Tuning tools (microbenchmarks, layout searches); not part of the hot path."""
