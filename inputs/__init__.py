"""Seeded synthetic inputs (generator + config recipes). Holds none of the method's arithmetic."""
