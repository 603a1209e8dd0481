"""Float64 CPU oracle of the batched drone-env step — TEST INFRASTRUCTURE (see drone_oracle.hpp)."""
