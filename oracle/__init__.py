"""oracle/ -- test infrastructure (plain fp64 CPU SHASTA written from the paper). Not the product."""
